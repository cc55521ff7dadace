// wcsim.cu -- the C ABI of include/wcsim.h: plan life cycle, argument checking, buffer ownership and the launch
// sequences.  All arithmetic of the path lives in raster.cu / convolve.cu / response.cu; there is no CPU fallback.
#include "../../include/wcsim.h"
#include "fft.cuh"
#include "internal.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace wcsim;

struct wcsim_plan {
    int n_wires = 0, n_ticks = 0, pad_w = 0, pad_t = 0, n_rw = 0, n_rt = 0, spec_stride = 0;
    double nsigma = 3.0;
    int scatter_mode = WCSIM_SCATTER_ATOMIC;
    cudaStream_t stream = nullptr;
    int device = 0, sm_count = 148;
    float *S = nullptr, *M = nullptr;
    float2 *spec = nullptr, *spec2 = nullptr, *Rhat = nullptr, *Rt = nullptr;
    float2 *spec_alloc = nullptr; // spec with its zero halo rows (wires_halo)
    float2 *tw_row = nullptr, *tw_real = nullptr, *tw_col = nullptr;
    int rt_rows = 0;
    int wire_mode = WCSIM_WIRES_AUTO;
    bool normalize = false; // renormalised patches (reading A24)
    int impact_K = 1;       // impact positions per wire (reading A25); S has s_wires = n_wires * impact_K fine rows
    int s_wires = 0;
    bool multi = false;     // created by wcsim_plan_create_planes
    bool capturing = false; // between wcsim_graph_begin and wcsim_graph_end
    unsigned long long captured_launches = 0;
    int live_graphs = 0;    // wcsim_graph objects that point at this plan (wcsim_plan_destroy refuses while > 0)
    short *dev_adc = nullptr; // ADC codes of wcsim_simulate_host_adc_async (allocated on first use)
    PlaneTable pt{};        // n = 1 for an ordinary plan
    Counters *counters = nullptr;
    float *amp_builtin = nullptr, *amp_custom = nullptr; // device, pad_t/2+1, scaled by pad_t^-1/2
    float *amp_armed = nullptr; // the armed custom spectrum's own copy (a later wcsim_add_noise must not change it)
    bool noise_armed = false;
    const float *armed_amp = nullptr;
    uint64_t armed_seed[kMaxPlanes] = {}; // plane p's noise seed (A26); a single-seed arm fills every entry alike
    TileScratch ts{};
    float *stage_block = nullptr; // device staging of the five host depo arrays, 5 * stage_cap floats
    long long stage_cap = 0;
    // profiling: CUDA events recorded around each stage on the plan's stream while enabled
    struct Span {
        cudaEvent_t beg, end;
        int stage;
    };
    int profiling = 0; // 0 off, WCSIM_PROFILE_KERNELS, WCSIM_PROFILE_CALLS
    std::vector<Span> pending;
    std::vector<cudaEvent_t> free_events;
    double stage_ms[WCSIM_N_STAGES] = {};
    unsigned long long stage_calls[WCSIM_N_STAGES] = {};
    unsigned long long launches = 0; // kernels of this library enqueued so far
};

namespace {

thread_local int tls_cuda_error = 0;

int fail_cuda(cudaError_t e)
{
    tls_cuda_error = (int)e;
    cudaGetLastError(); // clear the sticky-less error state
    return e == cudaErrorMemoryAllocation ? WCSIM_ENOMEM : WCSIM_ECUDA;
}

#define CU_TRY(expr)                                                                                                   \
    do {                                                                                                               \
        cudaError_t e__ = (expr);                                                                                      \
        if (e__ != cudaSuccess) return fail_cuda(e__);                                                                 \
    } while (0)

struct DeviceGuard {
    int prev = -1;
    bool ok = true;
    explicit DeviceGuard(int dev)
    {
        if (cudaGetDevice(&prev) != cudaSuccess) {
            ok = false;
            return;
        }
        if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
    }
    ~DeviceGuard()
    {
        int cur = -1;
        if (prev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != prev) cudaSetDevice(prev);
    }
};

cudaEvent_t take_event(wcsim_plan *p)
{
    cudaEvent_t e = nullptr;
    if (!p->free_events.empty()) {
        e = p->free_events.back();
        p->free_events.pop_back();
    } else if (cudaEventCreate(&e) != cudaSuccess) {
        e = nullptr;
    }
    return e;
}

// accumulate finished spans into stage_ms (synchronises the stream)
int harvest_spans(wcsim_plan *p)
{
    if (p->pending.empty()) return WCSIM_OK;
    CU_TRY(cudaStreamSynchronize(p->stream));
    for (auto &sp : p->pending) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, sp.beg, sp.end) == cudaSuccess) {
            p->stage_ms[sp.stage] += (double)ms;
            p->stage_calls[sp.stage] += 1;
        }
        p->free_events.push_back(sp.beg);
        p->free_events.push_back(sp.end);
    }
    p->pending.clear();
    return WCSIM_OK;
}

// RAII span: records an event pair around a stage when profiling is enabled
struct StageSpan {
    wcsim_plan *p;
    cudaEvent_t beg = nullptr, end = nullptr;
    int stage;
    StageSpan(wcsim_plan *plan, int st, bool enabled = true) : p(plan), stage(st)
    {
        if (!p->profiling || !enabled || p->capturing) return;
        if (p->pending.size() >= 8192) harvest_spans(p);
        beg = take_event(p);
        end = take_event(p);
        if (beg && end) cudaEventRecord(beg, p->stream);
    }
    ~StageSpan()
    {
        if (beg && end) {
            cudaEventRecord(end, p->stream);
            p->pending.push_back({beg, end, stage});
        }
    }
};

bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }
int next_pow2(long long n, int floor_)
{
    long long p = floor_;
    while (p < n) p <<= 1;
    return p > (1 << 30) ? 0 : (int)p;
}

// Wire axis of the convolution: direct summation over the response's wire offsets, or FFT / multiply / inverse FFT.
// Per output the direct form costs 4 n_rw FMAs, the FFT form a pad_w-point transform pair plus the read of Rhat.  AUTO
// takes the direct form up to the MEASURED crossover (profiles/r02_wire_crossover.md: both routes timed for response
// widths 21..129 at three plane sizes): direct wins up to 41 wires at pad_w = 1024 (FFT from 49), up to 97 at pad_w = 4096
// (FFT from 129), at 21 for pad_w = 512 (FFT from 41).
bool wires_direct(const wcsim_plan *p)
{
    if (p->wire_mode == WCSIM_WIRES_AUTO) {
        const int crossover = p->pad_w <= 512 ? 32 : p->pad_w <= 2048 ? 45 : 100;
        return p->multi || p->impact_K > 1 || p->n_rw <= crossover;
    }
    return p->wire_mode == WCSIM_WIRES_DIRECT;
}

ConvBuffers conv_buffers(const wcsim_plan *p)
{
    ConvBuffers b;
    b.S = p->S;
    b.M = p->M;
    b.spec = p->spec;
    b.spec2 = p->spec2;
    b.spec_inv = wires_direct(p) ? p->spec2 : p->spec;
    b.Rhat = p->Rhat;
    b.Rt = p->Rt;
    b.rt_rows = p->rt_rows;
    b.n_rw = p->n_rw;
    b.tw_row = p->tw_row;
    b.tw_real = p->tw_real;
    b.tw_col = p->tw_col;
    b.spec_stride = p->spec_stride;
    b.sm_count = p->sm_count;
    b.planes = p->pt;
    b.impact_K = p->impact_K;
    return b;
}

// denom > 0: flat table exp(-2 pi i j / denom), j < n.  denom = 0: the per-pass tables of fft.cuh for an n-point FFT.
int upload_twiddles(float2 **dev, int n, int denom, cudaStream_t st)
{
    std::vector<float2> h((size_t)(denom > 0 ? n : tw_size(n)));
    if (denom > 0) {
        for (int j = 0; j < n; ++j) {
            const double a = -2.0 * M_PI * (double)j / (double)denom;
            h[j] = make_float2((float)cos(a), (float)sin(a));
        }
    } else {
        build_pass_twiddles(n, h.data());
    }
    n = (int)h.size();
    CU_TRY(cudaMalloc((void **)dev, sizeof(float2) * (size_t)n));
    CU_TRY(cudaMemcpyAsync(*dev, h.data(), sizeof(float2) * (size_t)n, cudaMemcpyHostToDevice, st));
    CU_TRY(cudaStreamSynchronize(st));
    return WCSIM_OK;
}

// amplitude spectrum -> device, scaled by pad_t^-1/2 (orthonormal inverse transform, A15)
int upload_amp(wcsim_plan *p, const float *host_amp, float *dev)
{
    const int nk = p->pad_t / 2 + 1;
    std::vector<float> h((size_t)nk);
    const double scale = 1.0 / sqrt((double)p->pad_t);
    for (int k = 0; k < nk; ++k) {
        double a;
        if (host_amp) {
            a = (double)host_amp[k];
        } else { // A(f) = 3 (f/f0) exp(-f/f0), f0 = 0.1 f_Nyquist, f in cycles per tick (configs[3])
            const double f = (double)k / (double)p->pad_t, f0 = 0.1 * 0.5;
            a = 3.0 * (f / f0) * exp(-(f / f0));
        }
        h[k] = (float)(a * scale);
    }
    CU_TRY(cudaMemcpyAsync(dev, h.data(), sizeof(float) * (size_t)nk, cudaMemcpyHostToDevice, p->stream));
    CU_TRY(cudaStreamSynchronize(p->stream)); // h goes out of scope
    return WCSIM_OK;
}

int ensure_stage(wcsim_plan *p, long long n)
{
    if (n <= p->stage_cap) return WCSIM_OK;
    CU_TRY(cudaStreamSynchronize(p->stream));
    if (p->stage_block) cudaFree(p->stage_block);
    p->stage_block = nullptr;
    p->stage_cap = 0;
    const long long cap = n + n / 4 + 1024;
    CU_TRY(cudaMalloc((void **)&p->stage_block, sizeof(float) * 5 * (size_t)cap));
    p->stage_cap = cap;
    return WCSIM_OK;
}

// Deterministic sort-by-tile mode, all on the stream (no read-back): a depo is listed in the at most tile_max_listed()
// tiles its patch touches, so tile_max_listed() * n entries always suffice; a depo whose patch touches more tiles is not
// listed and goes through the atomic kernel into the same fixed-point grid (integer adds: the sum does not depend on the
// order), which tile_finalize folds into S.
int raster_tiled(wcsim_plan *p, GridDims g, DepoArrays d, long long n, uint64_t id_base, uint64_t seed, int fluctuate,
                 int *totals)
{
    TileScratch &ts = p->ts;
    const int n_tiles = ts.tiles_w * ts.tiles_t;
    const unsigned long long need = (unsigned long long)tile_max_listed() * (unsigned long long)n + 16ull;
    if (need > 0xFFFFFFFFull) return WCSIM_EINVAL; // 32-bit list offsets and depo indices: raster fewer depos per call
    if (need > ts.capacity) {
        if (p->capturing) return WCSIM_ESTATE; // grow the lists outside a capture: run the call once before
        CU_TRY(cudaStreamSynchronize(p->stream));
        if (ts.entries) cudaFree(ts.entries);
        ts.entries = nullptr;
        ts.capacity = 0;
        const unsigned long long cap = need + need / 4;
        CU_TRY(cudaMalloc((void **)&ts.entries, sizeof(unsigned int) * cap));
        ts.capacity = cap;
    }
    if (!ts.fix) { // first use of the fixed-point grid on this plan
        if (p->capturing) return WCSIM_ESTATE;
        const size_t bytes = sizeof(unsigned long long) * (size_t)g.n_wires * g.n_ticks;
        CU_TRY(cudaMalloc((void **)&ts.fix, bytes));
        CU_TRY(cudaMemsetAsync(ts.fix, 0, bytes, p->stream));
    }
    CU_TRY(cudaMemsetAsync(ts.tile_count, 0, sizeof(unsigned int) * (size_t)(n_tiles + 1), p->stream));
    CU_TRY(launch_tile_count(g, d, n, p->nsigma, ts, p->stream));
    CU_TRY(launch_tile_scan(ts, p->stream));
    CU_TRY(launch_tile_fill(g, d, n, p->nsigma, ts, p->stream));
    if (totals) CU_TRY(cudaMemsetAsync(totals, 0, sizeof(int) * (size_t)n, p->stream));
    CU_TRY(launch_count_invalid(d, n, p->counters, p->stream));
    CU_TRY(launch_tile_accumulate(g, d, id_base, seed, fluctuate, p->nsigma, ts, p->S, totals, p->counters, p->stream));
    CU_TRY(launch_raster_fixed(g, d, n, id_base, seed, fluctuate, p->nsigma, ts.fix, totals, p->counters, p->sm_count,
                               p->stream, true));
    CU_TRY(launch_tile_finalize(g, ts, p->S, p->stream));
    return WCSIM_OK;
}

int destroy_impl(wcsim_plan *p)
{
    int rc = WCSIM_OK;
    if (cudaStreamSynchronize(p->stream) != cudaSuccess) rc = fail_cuda(cudaGetLastError());
    void *bufs[] = {p->spec2,    p->Rt,
                    p->S,        p->M,           p->spec_alloc,  p->Rhat,           p->tw_row,        p->tw_real,
                    p->tw_col,   p->counters,    p->amp_builtin, p->amp_custom,     p->ts.tile_count, p->ts.tile_cursor,
                    p->amp_armed, p->dev_adc,
                    p->ts.entries, p->ts.slice_dev, p->ts.fix,  p->stage_block};
    for (void *b : bufs)
        if (b) cudaFree(b);
    for (auto &sp : p->pending) {
        cudaEventDestroy(sp.beg);
        cudaEventDestroy(sp.end);
    }
    for (cudaEvent_t e : p->free_events) cudaEventDestroy(e);
    delete p;
    return rc;
}

} // namespace

namespace {

// plan creation for 1..kMaxPlanes planes stacked along the wire axis (same n_ticks, padding and response footprint).
// `multi`: created by wcsim_plan_create_planes (direct wire pass only, no Rhat)
int create_impl(wcsim_plan **out, int n_planes, const int *plane_wires, int n_ticks, const float *const *responses,
                int n_rwires, int n_rticks, wcsim_pad pad, float nsigma, int scatter_mode, void *cuda_stream, bool multi,
                int K = 1)
{
    if (!out) return WCSIM_EINVAL;
    *out = nullptr;
    if (K < 1 || K > 64 || (K > 1 && (multi || n_planes != 1))) return WCSIM_EINVAL;
    if (!plane_wires || !responses || n_planes < 1 || n_planes > kMaxPlanes || n_ticks <= 0 || n_rwires <= 0 ||
        n_rticks <= 0 || (n_rwires % 2) == 0)
        return WCSIM_EINVAL;
    long long total_wires = 0;
    int max_wires = 0;
    for (int p = 0; p < n_planes; ++p) {
        if (plane_wires[p] <= 0 || !responses[p]) return WCSIM_EINVAL;
        total_wires += plane_wires[p];
        max_wires = plane_wires[p] > max_wires ? plane_wires[p] : max_wires;
    }
    for (int k = 1; k < K; ++k)
        if (!responses[k]) return WCSIM_EINVAL; // K > 1: responses[k] is the response of impact position k
    if (!(nsigma > 0.0f) || !std::isfinite(nsigma)) return WCSIM_EINVAL;
    if (scatter_mode < WCSIM_SCATTER_ATOMIC || scatter_mode > WCSIM_SCATTER_FIXED) return WCSIM_EINVAL;
    if (multi && scatter_mode == WCSIM_SCATTER_TILED) return WCSIM_EINVAL; // tiles belong to one plane
    if (pad.wires < 0 || pad.ticks < 0) return WCSIM_EINVAL;
    const int c = (n_rwires - 1) / 2;
    const long long need_t = (long long)n_ticks + n_rticks - 1, need_w = (long long)max_wires + c;
    const int pad_t = pad.ticks ? pad.ticks : next_pow2(need_t, 32);
    // automatic wire padding also keeps the wrapped response from overlapping itself (pad_w >= n_rwires)
    const int pad_w = (pad.wires && !multi) ? pad.wires : next_pow2(need_w > n_rwires ? need_w : (long long)n_rwires, 16);
    if (!is_pow2(pad_t) || !is_pow2(pad_w) || pad_t < need_t || pad_w < need_w || pad_t < 32 || pad_w < 16)
        return WCSIM_EINVAL;
    if (pad_w < n_rwires) return WCSIM_EINVAL; // the wrapped response must not overlap itself
    if (!conv_sizes_supported(pad_w, pad_t)) return WCSIM_EINVAL;
    if (total_wires * K * n_ticks >= (1ll << 30)) return WCSIM_EINVAL; // bin index + 2 flag bits in 32 (draw queues)
    const int n_wires = (int)total_wires;
    const int s_wires = n_wires * K; // rows of S and of the row spectra

    int dev = 0;
    CU_TRY(cudaGetDevice(&dev));
    wcsim_plan *p = new (std::nothrow) wcsim_plan;
    if (!p) return WCSIM_ENOMEM;
    p->n_wires = n_wires;
    p->n_ticks = n_ticks;
    p->pad_w = pad_w;
    p->pad_t = pad_t;
    p->n_rw = n_rwires;
    p->n_rt = n_rticks;
    p->spec_stride = pad_t / 2 + 8;
    p->nsigma = (double)nsigma;
    p->scatter_mode = scatter_mode;
    p->stream = (cudaStream_t)cuda_stream;
    p->device = dev;
    p->multi = multi;
    p->impact_K = K;
    p->s_wires = s_wires;
    if (multi || K > 1) p->wire_mode = WCSIM_WIRES_DIRECT;

    // the plane table: stacked rows, halo rows of the row spectra between the planes, row groups of the wire pass
    int halo_lo = 0, halo_hi = 0;
    wires_halo(n_rwires, &halo_lo, &halo_hi);
    halo_lo *= K; // fine rows
    halo_hi = halo_hi * K + (K - 1);
    const int per_group = wires_rows_per_group();
    PlaneTable &pt = p->pt;
    pt.n = n_planes;
    int row = 0, srow = 0, grp = 0;
    for (int q = 0; q < n_planes; ++q) {
        pt.row0[q] = row;
        pt.srow0[q] = srow + q * (halo_lo + halo_hi); // relative to `spec`, which starts after the first low halo
        pt.grp0[q] = grp;
        row += plane_wires[q];
        srow += plane_wires[q];
        grp += (plane_wires[q] + per_group - 1) / per_group;
    }
    for (int q = n_planes; q <= kMaxPlanes; ++q) pt.row0[q] = row, pt.grp0[q] = grp;
    for (int q = n_planes; q < kMaxPlanes; ++q) pt.srow0[q] = 0;

    float *dev_R = nullptr;
    double2 *dev_tmp = nullptr;
    int rc = [&]() -> int {
        CU_TRY(cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, dev));
        const size_t grid = (size_t)n_wires * n_ticks, sgrid = (size_t)s_wires * n_ticks;
        CU_TRY(cudaMalloc((void **)&p->S, sizeof(float) * sgrid));
        CU_TRY(cudaMalloc((void **)&p->M, sizeof(float) * grid));
        const size_t spec_rows = (size_t)s_wires + (size_t)n_planes * (halo_lo + halo_hi);
        CU_TRY(cudaMalloc((void **)&p->spec_alloc, sizeof(float2) * spec_rows * p->spec_stride));
        p->spec = p->spec_alloc + (size_t)halo_lo * p->spec_stride;
        CU_TRY(cudaMalloc((void **)&p->spec2, sizeof(float2) * (size_t)n_wires * p->spec_stride));
        const bool want_rhat = !multi && K == 1;
        if (want_rhat) CU_TRY(cudaMalloc((void **)&p->Rhat, sizeof(float2) * (size_t)pad_w * p->spec_stride));
        p->rt_rows = (n_rwires + wires_chunk() - 1) / wires_chunk() * wires_chunk();
        const int n_resp = n_planes * K; // response blocks: one per plane, or one per impact position
        CU_TRY(cudaMalloc((void **)&p->Rt, sizeof(float2) * (size_t)n_resp * p->rt_rows * p->spec_stride));
        CU_TRY(cudaMalloc((void **)&p->counters, sizeof(Counters)));
        CU_TRY(cudaMalloc((void **)&p->amp_builtin, sizeof(float) * (size_t)(pad_t / 2 + 1)));
        CU_TRY(cudaMalloc((void **)&p->amp_custom, sizeof(float) * (size_t)(pad_t / 2 + 1)));
        CU_TRY(cudaMalloc((void **)&p->amp_armed, sizeof(float) * (size_t)(pad_t / 2 + 1)));
        CU_TRY(cudaMemsetAsync(p->S, 0, sizeof(float) * sgrid, p->stream));
        CU_TRY(cudaMemsetAsync(p->M, 0, sizeof(float) * grid, p->stream));
        CU_TRY(cudaMemsetAsync(p->spec_alloc, 0, sizeof(float2) * spec_rows * p->spec_stride, p->stream));
        CU_TRY(cudaMemsetAsync(p->spec2, 0, sizeof(float2) * (size_t)n_wires * p->spec_stride, p->stream));
        CU_TRY(cudaMemsetAsync(p->counters, 0, sizeof(Counters), p->stream));
        int r = upload_twiddles(&p->tw_row, pad_t / 2, 0, p->stream);
        if (r) return r;
        r = upload_twiddles(&p->tw_real, pad_t / 2, pad_t, p->stream);
        if (r) return r;
        r = upload_twiddles(&p->tw_col, pad_w, 0, p->stream);
        if (r) return r;
        r = upload_amp(p, nullptr, p->amp_builtin);
        if (r) return r;
        // tile lists of the deterministic scatter mode
        tile_shape(&p->ts.tile_w, &p->ts.tile_t);
        p->ts.tiles_w = (s_wires + p->ts.tile_w - 1) / p->ts.tile_w;
        p->ts.tiles_t = (n_ticks + p->ts.tile_t - 1) / p->ts.tile_t;
        const size_t n_tiles = (size_t)p->ts.tiles_w * p->ts.tiles_t;
        CU_TRY(cudaMalloc((void **)&p->ts.tile_count, sizeof(unsigned int) * (n_tiles + 1)));
        CU_TRY(cudaMalloc((void **)&p->ts.tile_cursor, sizeof(unsigned int) * n_tiles));
        CU_TRY(cudaMalloc((void **)&p->ts.slice_dev, sizeof(unsigned int)));
        // response spectra: Rt of every plane (direct wire pass), Rhat of a single-plane plan (FFT wire pass)
        const size_t nr = (size_t)n_rwires * n_rticks;
        CU_TRY(cudaMalloc((void **)&dev_R, sizeof(float) * nr));
        CU_TRY(cudaMalloc((void **)&dev_tmp, sizeof(double2) * (size_t)n_rwires * (pad_t / 2 + 1)));
        for (int q = 0; q < n_resp; ++q) {
            CU_TRY(cudaMemcpyAsync(dev_R, responses[q], sizeof(float) * nr, cudaMemcpyHostToDevice, p->stream));
            CU_TRY(build_response_spectrum(dev_R, n_rwires, n_rticks, pad_w, pad_t, p->spec_stride, dev_tmp, p->Rhat,
                                           p->stream));
            CU_TRY(build_response_rows(dev_tmp, n_rwires, p->rt_rows, pad_t, p->spec_stride,
                                       p->Rt + (size_t)q * p->rt_rows * p->spec_stride, p->stream));
            CU_TRY(cudaStreamSynchronize(p->stream)); // responses[q] may be pageable; dev_R is reused
        }
        CU_TRY(conv_configure(pad_w, pad_t));
        CU_TRY(raster_configure(p->stream));
        CU_TRY(cudaStreamSynchronize(p->stream));
        return WCSIM_OK;
    }();
    if (dev_R) cudaFree(dev_R);
    if (dev_tmp) cudaFree(dev_tmp);
    if (rc != WCSIM_OK) {
        const int keep = tls_cuda_error;
        destroy_impl(p);
        tls_cuda_error = keep;
        return rc;
    }
    *out = p;
    return WCSIM_OK;
}

} // namespace

extern "C" {

int wcsim_plan_create(wcsim_plan **out, int n_wires, int n_ticks, const float *response, int n_rwires, int n_rticks,
                      wcsim_pad pad, float nsigma, int scatter_mode, void *cuda_stream)
{
    if (out) *out = nullptr;
    return create_impl(out, 1, &n_wires, n_ticks, &response, n_rwires, n_rticks, pad, nsigma, scatter_mode, cuda_stream,
                       false);
}

int wcsim_plan_create_impact(wcsim_plan **out, int n_wires, int n_ticks, int n_impact, const float *const *responses,
                             int n_rwires, int n_rticks, int pad_ticks, float nsigma, int scatter_mode, void *cuda_stream)
{
    if (out) *out = nullptr;
    wcsim_pad pad;
    pad.wires = 0;
    pad.ticks = pad_ticks;
    return create_impl(out, 1, &n_wires, n_ticks, responses, n_rwires, n_rticks, pad, nsigma, scatter_mode, cuda_stream,
                       false, n_impact);
}

int wcsim_get_charge_dims(const wcsim_plan *plan, int *rows, int *n_ticks, int *n_impact)
{
    if (!plan) return WCSIM_EINVAL;
    if (rows) *rows = plan->s_wires;
    if (n_ticks) *n_ticks = plan->n_ticks;
    if (n_impact) *n_impact = plan->impact_K;
    return WCSIM_OK;
}

int wcsim_plan_create_planes(wcsim_plan **out, int n_planes, const int *n_wires, int n_ticks,
                             const float *const *responses, int n_rwires, int n_rticks, int pad_ticks, float nsigma,
                             int scatter_mode, void *cuda_stream)
{
    if (out) *out = nullptr;
    wcsim_pad pad;
    pad.wires = 0;
    pad.ticks = pad_ticks;
    return create_impl(out, n_planes, n_wires, n_ticks, responses, n_rwires, n_rticks, pad, nsigma, scatter_mode,
                       cuda_stream, true);
}

int wcsim_raster_scatter(wcsim_plan *plan, const wcsim_depos *depos, long long n, unsigned long long depo_id_base,
                         unsigned long long seed, int fluctuate, int *dev_depo_totals)
{
    if (!plan || n < 0 || fluctuate < 0 || fluctuate > 2) return WCSIM_EINVAL;
    if (plan->multi) return WCSIM_ESTATE; // a multi-plane plan is rastered by wcsim_raster_scatter_planes
    if (n == 0) return WCSIM_OK;
    if (!depos || !depos->t0 || !depos->x0 || !depos->sigma_t || !depos->sigma_x || !depos->q) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    if (!guard.ok) return fail_cuda(cudaGetLastError());
    const GridDims g{plan->s_wires, plan->n_ticks}; // the charge grid: n_wires * impact_K rows
    const DepoArrays d{depos->t0, depos->x0, depos->sigma_t, depos->sigma_x, depos->q};
    if (plan->normalize) fluctuate |= kRasterNormalize; // internal.h: flag bit of the launchers' `fluctuate`
    StageSpan span(plan, WCSIM_STAGE_RASTER);
    if (plan->scatter_mode == WCSIM_SCATTER_TILED) {
        const int rc = raster_tiled(plan, g, d, n, depo_id_base, seed, fluctuate, dev_depo_totals);
        if (rc == WCSIM_OK) plan->launches += 7;
        return rc;
    }
    if (dev_depo_totals) CU_TRY(cudaMemsetAsync(dev_depo_totals, 0, sizeof(int) * (size_t)n, plan->stream));
    const bool fixed = plan->scatter_mode == WCSIM_SCATTER_FIXED;
    if (fixed && !plan->ts.fix) { // first use of the fixed-point grid on this plan
        if (plan->capturing) return WCSIM_ESTATE; // allocate before capturing: run the call once outside the capture
        const size_t bytes = sizeof(unsigned long long) * (size_t)g.n_wires * g.n_ticks;
        CU_TRY(cudaMalloc((void **)&plan->ts.fix, bytes));
        CU_TRY(cudaMemsetAsync(plan->ts.fix, 0, bytes, plan->stream));
    }
    // the draw queues index per-depo totals with 32 bits: with totals requested, launch 2^31 depos at a time
    const long long chunk = dev_depo_totals ? (1ll << 31) : n;
    for (long long first = 0; first < n; first += chunk) {
        const long long m = n - first < chunk ? n - first : chunk;
        const DepoArrays dc{d.t0 + first, d.x0 + first, d.sigma_t + first, d.sigma_x + first, d.q + first};
        plan->launches += 1;
        if (fixed)
            CU_TRY(launch_raster_fixed(g, dc, m, depo_id_base + (unsigned long long)first, seed, fluctuate, plan->nsigma,
                                       plan->ts.fix, dev_depo_totals ? dev_depo_totals + first : nullptr, plan->counters,
                                       plan->sm_count, plan->stream));
        else
            CU_TRY(launch_raster_atomic(g, dc, m, depo_id_base + (unsigned long long)first, seed, fluctuate, plan->nsigma,
                                        plan->S, dev_depo_totals ? dev_depo_totals + first : nullptr, plan->counters,
                                        plan->sm_count, plan->stream));
    }
    if (fixed) {
        plan->launches += 1;
        CU_TRY(launch_tile_finalize(g, plan->ts, plan->S, plan->stream));
    }
    return WCSIM_OK;
}

namespace {
int raster_scatter_planes_impl(wcsim_plan *plan, const wcsim_depos *depos, const long long *n,
                               const unsigned long long *seeds, int n_seeds, int fluctuate);
}

int wcsim_raster_scatter_planes(wcsim_plan *plan, const wcsim_depos *depos, const long long *n, unsigned long long seed,
                                int fluctuate)
{
    return raster_scatter_planes_impl(plan, depos, n, &seed, 1, fluctuate);
}

int wcsim_raster_scatter_planes_seeded(wcsim_plan *plan, const wcsim_depos *depos, const long long *n,
                                       const unsigned long long *seeds, int fluctuate)
{
    if (!plan || !seeds) return WCSIM_EINVAL;
    return raster_scatter_planes_impl(plan, depos, n, seeds, plan->pt.n, fluctuate);
}

namespace {
int raster_scatter_planes_impl(wcsim_plan *plan, const wcsim_depos *depos, const long long *n,
                               const unsigned long long *seeds, int n_seeds, int fluctuate)
{
    if (!plan || !depos || !n || fluctuate < 0 || fluctuate > 2) return WCSIM_EINVAL;
    if (plan->scatter_mode == WCSIM_SCATTER_TILED) return WCSIM_ESTATE;
    DeviceGuard guard(plan->device);
    if (!guard.ok) return fail_cuda(cudaGetLastError());
    RasterPlanes rp{};
    rp.n = plan->pt.n;
    const int per_batch = raster_batch_depos();
    long long batches = 0;
    for (int p = 0; p < rp.n; ++p) {
        if (n[p] < 0) return WCSIM_EINVAL;
        if (n[p] > 0 && (!depos[p].t0 || !depos[p].x0 || !depos[p].sigma_t || !depos[p].sigma_x || !depos[p].q))
            return WCSIM_EINVAL;
        rp.d[p] = DepoArrays{depos[p].t0, depos[p].x0, depos[p].sigma_t, depos[p].sigma_x, depos[p].q};
        rp.count[p] = n[p];
        rp.seed[p] = seeds[p < n_seeds ? p : n_seeds - 1];
        rp.batch0[p] = batches;
        batches += (n[p] + per_batch - 1) / per_batch;
        rp.n_wires[p] = plan->impact_K > 1 ? plan->s_wires : plan->pt.row0[p + 1] - plan->pt.row0[p];
        rp.row0[p] = plan->pt.row0[p];
    }
    for (int p = rp.n; p <= kMaxPlanes; ++p) rp.batch0[p] = batches;
    if (batches == 0) return WCSIM_OK;
    if (plan->normalize) fluctuate |= kRasterNormalize;
    StageSpan span(plan, WCSIM_STAGE_RASTER);
    const bool fixed = plan->scatter_mode == WCSIM_SCATTER_FIXED;
    if (fixed && !plan->ts.fix) { // first use of the fixed-point grid on this plan
        if (plan->capturing) return WCSIM_ESTATE;
        const size_t bytes = sizeof(unsigned long long) * (size_t)plan->s_wires * plan->n_ticks;
        CU_TRY(cudaMalloc((void **)&plan->ts.fix, bytes));
        CU_TRY(cudaMemsetAsync(plan->ts.fix, 0, bytes, plan->stream));
    }
    plan->launches += 1;
    CU_TRY(launch_raster_planes(plan->n_ticks, rp, fluctuate, plan->nsigma,
                                fixed ? (void *)plan->ts.fix : (void *)plan->S, fixed, plan->counters, plan->sm_count,
                                plan->stream));
    if (fixed) {
        plan->launches += 1;
        CU_TRY(launch_tile_finalize(GridDims{plan->s_wires, plan->n_ticks}, plan->ts, plan->S, plan->stream));
    }
    return WCSIM_OK;
}
} // namespace

int wcsim_get_plane_rows(const wcsim_plan *plan, int plane, int *first_row, int *n_rows)
{
    if (!plan || plane < 0 || plane >= plan->pt.n) return WCSIM_EINVAL;
    if (first_row) *first_row = plan->pt.row0[plane];
    if (n_rows) *n_rows = plan->pt.row0[plane + 1] - plan->pt.row0[plane];
    return WCSIM_OK;
}

int wcsim_convolve(wcsim_plan *plan)
{
    if (!plan) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    if (!guard.ok) return fail_cuda(cudaGetLastError());
    const GridDims g{plan->n_wires, plan->n_ticks};
    const ConvBuffers b = conv_buffers(plan);
    NoiseArgs nz{};
    if (plan->noise_armed) {
        nz = noise_args(plan->armed_amp, plan->armed_seed, kMaxPlanes);
        plan->noise_armed = false;
    }
    const bool per_kernel = plan->profiling == WCSIM_PROFILE_KERNELS;
    StageSpan whole(plan, WCSIM_STAGE_CONVOLVE, !per_kernel);
    {
        StageSpan span(plan, WCSIM_STAGE_ROWS_FORWARD, per_kernel);
        CU_TRY(launch_rows_forward(GridDims{plan->s_wires, plan->n_ticks}, plan->pad_t, b, plan->stream));
    }
    {
        StageSpan span(plan, WCSIM_STAGE_COLS, per_kernel);
        if (wires_direct(plan))
            CU_TRY(launch_wires(g, plan->pad_t, b, plan->stream));
        else
            CU_TRY(launch_cols(g, plan->pad_w, plan->pad_t, b, plan->stream));
    }
    {
        StageSpan span(plan, WCSIM_STAGE_ROWS_INVERSE, per_kernel);
        CU_TRY(launch_rows_inverse(g, plan->pad_t, b, nz, true, false, plan->stream));
    }
    plan->launches += 3;
    return WCSIM_OK;
}

static int noise_amp_ptr(wcsim_plan *plan, const float *amp, const float **dev)
{
    if (!amp) {
        *dev = plan->amp_builtin;
        return WCSIM_OK;
    }
    const int rc = upload_amp(plan, amp, plan->amp_custom);
    *dev = plan->amp_custom;
    return rc;
}

namespace {
int add_noise_impl(wcsim_plan *plan, const float *amp, const unsigned long long *seeds, int n_seeds)
{
    if (!plan) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    if (!guard.ok) return fail_cuda(cudaGetLastError());
    if (amp && plan->capturing) return WCSIM_ESTATE; // the upload synchronises
    const float *dev_amp = nullptr;
    const int rc = noise_amp_ptr(plan, amp, &dev_amp);
    if (rc) return rc;
    static_assert(sizeof(unsigned long long) == sizeof(uint64_t), "seed width");
    const NoiseArgs nz = noise_args(dev_amp, reinterpret_cast<const uint64_t *>(seeds), n_seeds);
    const GridDims g{plan->n_wires, plan->n_ticks};
    StageSpan span(plan, WCSIM_STAGE_NOISE);
    CU_TRY(launch_rows_inverse(g, plan->pad_t, conv_buffers(plan), nz, false, true, plan->stream));
    plan->launches += 1;
    return WCSIM_OK;
}

int arm_noise_impl(wcsim_plan *plan, const float *amp, const unsigned long long *seeds, int n_seeds)
{
    if (!plan) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    if (!guard.ok) return fail_cuda(cudaGetLastError());
    if (amp && plan->capturing) return WCSIM_ESTATE; // the upload synchronises
    const float *dev = plan->amp_builtin;
    if (amp) { // the armed spectrum gets its own device copy: a later wcsim_add_noise(amp') must not change it
        const int rc = upload_amp(plan, amp, plan->amp_armed);
        if (rc) return rc;
        dev = plan->amp_armed;
    }
    plan->armed_amp = dev;
    for (int p = 0; p < kMaxPlanes; ++p) plan->armed_seed[p] = seeds[p < n_seeds ? p : n_seeds - 1];
    plan->noise_armed = true;
    return WCSIM_OK;
}
} // namespace

int wcsim_add_noise(wcsim_plan *plan, const float *amp, unsigned long long seed) { return add_noise_impl(plan, amp, &seed, 1); }
int wcsim_arm_noise(wcsim_plan *plan, const float *amp, unsigned long long seed) { return arm_noise_impl(plan, amp, &seed, 1); }
int wcsim_add_noise_planes(wcsim_plan *plan, const float *amp, const unsigned long long *seeds)
{
    if (!plan || !seeds) return WCSIM_EINVAL;
    return add_noise_impl(plan, amp, seeds, plan->pt.n);
}
int wcsim_arm_noise_planes(wcsim_plan *plan, const float *amp, const unsigned long long *seeds)
{
    if (!plan || !seeds) return WCSIM_EINVAL;
    return arm_noise_impl(plan, amp, seeds, plan->pt.n);
}

int wcsim_plan_destroy(wcsim_plan *plan)
{
    if (!plan) return WCSIM_OK;
    if (plan->live_graphs > 0) return WCSIM_ESTATE; // its graphs hold a pointer to it: destroy them first
    DeviceGuard guard(plan->device);
    return destroy_impl(plan);
}

int wcsim_clear(wcsim_plan *plan)
{
    if (!plan) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    CU_TRY(launch_clear(plan->S, (long long)plan->s_wires * plan->n_ticks, plan->sm_count, plan->stream));
    plan->launches += 1;
    return WCSIM_OK;
}

int wcsim_clear_output(wcsim_plan *plan)
{
    if (!plan) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    CU_TRY(cudaMemsetAsync(plan->M, 0, sizeof(float) * (size_t)plan->n_wires * plan->n_ticks, plan->stream));
    return WCSIM_OK;
}

int wcsim_sync(wcsim_plan *plan)
{
    if (!plan) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    CU_TRY(cudaStreamSynchronize(plan->stream));
    return WCSIM_OK;
}

int wcsim_set_scatter_mode(wcsim_plan *plan, int scatter_mode)
{
    if (!plan || scatter_mode < WCSIM_SCATTER_ATOMIC || scatter_mode > WCSIM_SCATTER_FIXED) return WCSIM_EINVAL;
    plan->scatter_mode = scatter_mode;
    return WCSIM_OK;
}

int wcsim_get_wire_mode(const wcsim_plan *plan, int *resolved)
{
    if (!plan || !resolved) return WCSIM_EINVAL;
    *resolved = wires_direct(plan) ? WCSIM_WIRES_DIRECT : WCSIM_WIRES_FFT;
    return WCSIM_OK;
}

int wcsim_set_normalize(wcsim_plan *plan, int on)
{
    if (!plan) return WCSIM_EINVAL;
    plan->normalize = on != 0;
    return WCSIM_OK;
}

int wcsim_set_wire_mode(wcsim_plan *plan, int wire_mode)
{
    if (!plan || wire_mode < WCSIM_WIRES_AUTO || wire_mode > WCSIM_WIRES_DIRECT) return WCSIM_EINVAL;
    const bool direct_only = plan->multi || plan->impact_K > 1; // stacked planes, impact positions: direct wire pass only
    if (direct_only && wire_mode == WCSIM_WIRES_FFT) return WCSIM_ESTATE;
    if (direct_only) wire_mode = WCSIM_WIRES_DIRECT;
    plan->wire_mode = wire_mode;
    return WCSIM_OK;
}

int wcsim_charge_ptr(wcsim_plan *plan, float **dev)
{
    if (!plan || !dev) return WCSIM_EINVAL;
    *dev = plan->S;
    return WCSIM_OK;
}

int wcsim_output_ptr(wcsim_plan *plan, float **dev)
{
    if (!plan || !dev) return WCSIM_EINVAL;
    *dev = plan->M;
    return WCSIM_OK;
}

int wcsim_get_dims(const wcsim_plan *plan, int *n_wires, int *n_ticks, int *pad_wires, int *pad_ticks)
{
    if (!plan) return WCSIM_EINVAL;
    if (n_wires) *n_wires = plan->n_wires;
    if (n_ticks) *n_ticks = plan->n_ticks;
    if (pad_wires) *pad_wires = plan->pad_w;
    if (pad_ticks) *pad_ticks = plan->pad_t;
    return WCSIM_OK;
}

int wcsim_get_stats(wcsim_plan *plan, wcsim_stats *out)
{
    if (!plan || !out) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    Counters c;
    CU_TRY(cudaMemcpyAsync(&c, plan->counters, sizeof(c), cudaMemcpyDeviceToHost, plan->stream));
    CU_TRY(cudaStreamSynchronize(plan->stream));
    out->depos_skipped = c.depos_skipped;
    out->bins_drawn = c.bins_drawn;
    return WCSIM_OK;
}

int wcsim_reset_stats(wcsim_plan *plan)
{
    if (!plan) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    CU_TRY(cudaMemsetAsync(plan->counters, 0, sizeof(Counters), plan->stream));
    return WCSIM_OK;
}

namespace {

// copies the depos in, runs the plane-event, copies M (host_M) or its ADC codes (host_adc) out; everything enqueued
int simulate_host_impl(wcsim_plan *plan, const float *const host[5], long long n, unsigned long long seed, int fluctuate,
                       int noise, unsigned long long noise_seed, float *host_M, short *host_adc, float gain, float baseline,
                       int bits)
{
    if (!plan || n < 0 || (!host_M && !host_adc) || plan->multi) return plan && plan->multi ? WCSIM_ESTATE : WCSIM_EINVAL;
    if (n > 0 && (!host[0] || !host[1] || !host[2] || !host[3] || !host[4])) return WCSIM_EINVAL;
    if (host_adc && (bits < 1 || bits > 15)) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    if (!guard.ok) return fail_cuda(cudaGetLastError());
    int rc = ensure_stage(plan, n);
    if (rc) return rc;
    const size_t grid = (size_t)plan->n_wires * plan->n_ticks;
    if (host_adc && !plan->dev_adc) CU_TRY(cudaMalloc((void **)&plan->dev_adc, sizeof(short) * ((grid + 3) / 4 * 4)));
    float *dev[5];
    for (int a = 0; a < 5; ++a) dev[a] = plan->stage_block + (size_t)a * (size_t)n;
    // five arrays that follow one another in host memory (one pinned block) go over in one copy
    bool contiguous = n > 0;
    for (int a = 1; a < 5 && contiguous; ++a) contiguous = host[a] == host[a - 1] + n;
    if (contiguous) {
        CU_TRY(cudaMemcpyAsync(dev[0], host[0], sizeof(float) * 5 * (size_t)n, cudaMemcpyHostToDevice, plan->stream));
    } else {
        for (int a = 0; a < 5 && n > 0; ++a)
            CU_TRY(cudaMemcpyAsync(dev[a], host[a], sizeof(float) * (size_t)n, cudaMemcpyHostToDevice, plan->stream));
    }
    rc = wcsim_clear(plan);
    if (rc) return rc;
    const wcsim_depos d{dev[0], dev[1], dev[2], dev[3], dev[4]};
    rc = wcsim_raster_scatter(plan, &d, n, 0ull, seed, fluctuate, nullptr);
    if (rc) return rc;
    if (noise) {
        rc = wcsim_arm_noise(plan, nullptr, noise_seed);
        if (rc) return rc;
    }
    rc = wcsim_convolve(plan);
    if (rc) return rc;
    if (host_adc) {
        rc = wcsim_digitize(plan, gain, baseline, bits, plan->dev_adc);
        if (rc) return rc;
        CU_TRY(cudaMemcpyAsync(host_adc, plan->dev_adc, sizeof(short) * grid, cudaMemcpyDeviceToHost, plan->stream));
    }
    if (host_M) CU_TRY(cudaMemcpyAsync(host_M, plan->M, sizeof(float) * grid, cudaMemcpyDeviceToHost, plan->stream));
    return WCSIM_OK;
}

} // namespace

int wcsim_simulate_host_async(wcsim_plan *plan, const float *host_t0, const float *host_x0, const float *host_sigma_t,
                        const float *host_sigma_x, const float *host_q, long long n, unsigned long long seed,
                        int fluctuate, int noise, unsigned long long noise_seed, float *host_M)
{
    if (!host_M) return WCSIM_EINVAL;
    const float *const host[5] = {host_t0, host_x0, host_sigma_t, host_sigma_x, host_q};
    return simulate_host_impl(plan, host, n, seed, fluctuate, noise, noise_seed, host_M, nullptr, 0.f, 0.f, 0);
}

int wcsim_simulate_host_adc_async(wcsim_plan *plan, const float *host_t0, const float *host_x0, const float *host_sigma_t,
                                  const float *host_sigma_x, const float *host_q, long long n, unsigned long long seed,
                                  int fluctuate, int noise, unsigned long long noise_seed, float gain, float baseline,
                                  int bits, short *host_adc)
{
    if (!host_adc) return WCSIM_EINVAL;
    const float *const host[5] = {host_t0, host_x0, host_sigma_t, host_sigma_x, host_q};
    return simulate_host_impl(plan, host, n, seed, fluctuate, noise, noise_seed, nullptr, host_adc, gain, baseline, bits);
}

int wcsim_simulate_host(wcsim_plan *plan, const float *host_t0, const float *host_x0, const float *host_sigma_t,
                        const float *host_sigma_x, const float *host_q, long long n, unsigned long long seed,
                        int fluctuate, int noise, unsigned long long noise_seed, float *host_M)
{
    const int rc = wcsim_simulate_host_async(plan, host_t0, host_x0, host_sigma_t, host_sigma_x, host_q, n, seed,
                                             fluctuate, noise, noise_seed, host_M);
    if (rc) return rc;
    DeviceGuard guard(plan->device);
    if (!guard.ok) return fail_cuda(cudaGetLastError());
    CU_TRY(cudaStreamSynchronize(plan->stream));
    return WCSIM_OK;
}

// ---- CUDA graphs: a launch sequence captured once and replayed ----
struct wcsim_graph {
    wcsim_plan *plan;
    cudaGraph_t graph;
    cudaGraphExec_t exec;
    unsigned long long launches; // kernels of this library inside one replay
};

int wcsim_graph_begin(wcsim_plan *plan)
{
    if (!plan) return WCSIM_EINVAL;
    if (plan->capturing || plan->stream == nullptr) return WCSIM_ESTATE; // the legacy default stream cannot be captured
    DeviceGuard guard(plan->device);
    if (!guard.ok) return fail_cuda(cudaGetLastError());
    const int rc = harvest_spans(plan);
    if (rc) return rc;
    CU_TRY(cudaStreamBeginCapture(plan->stream, cudaStreamCaptureModeRelaxed));
    plan->capturing = true;
    plan->captured_launches = plan->launches;
    return WCSIM_OK;
}

int wcsim_graph_end(wcsim_plan *plan, wcsim_graph **out)
{
    if (out) *out = nullptr;
    if (!plan || !out) return WCSIM_EINVAL;
    if (!plan->capturing) return WCSIM_ESTATE;
    DeviceGuard guard(plan->device);
    plan->capturing = false;
    const unsigned long long inside = plan->launches - plan->captured_launches;
    plan->launches = plan->captured_launches; // nothing ran yet
    cudaGraph_t g = nullptr;
    CU_TRY(cudaStreamEndCapture(plan->stream, &g));
    if (!g) return WCSIM_ECUDA;
    cudaGraphExec_t exec = nullptr;
    const cudaError_t e = cudaGraphInstantiate(&exec, g, 0);
    if (e != cudaSuccess) {
        cudaGraphDestroy(g);
        return fail_cuda(e);
    }
    wcsim_graph *gr = new (std::nothrow) wcsim_graph{plan, g, exec, inside};
    if (!gr) {
        cudaGraphExecDestroy(exec);
        cudaGraphDestroy(g);
        return WCSIM_ENOMEM;
    }
    plan->live_graphs += 1;
    *out = gr;
    return WCSIM_OK;
}

int wcsim_graph_update(wcsim_plan *plan, wcsim_graph *graph)
{
    if (!plan || !graph) return WCSIM_EINVAL;
    if (!plan->capturing || graph->plan != plan) return WCSIM_ESTATE;
    DeviceGuard guard(plan->device);
    plan->capturing = false;
    const unsigned long long inside = plan->launches - plan->captured_launches;
    plan->launches = plan->captured_launches; // nothing ran yet
    cudaGraph_t g = nullptr;
    CU_TRY(cudaStreamEndCapture(plan->stream, &g));
    if (!g) return WCSIM_ECUDA;
    cudaGraphExecUpdateResultInfo info{};
    const cudaError_t e = cudaGraphExecUpdate(graph->exec, g, &info);
    if (e != cudaSuccess) {
        cudaGraphDestroy(g);
        if (e == cudaErrorGraphExecUpdateFailure) { // not the same sequence of calls as the one the graph was made from
            cudaGetLastError();
            return WCSIM_ESTATE;
        }
        return fail_cuda(e);
    }
    cudaGraphDestroy(graph->graph);
    graph->graph = g;
    graph->launches = inside;
    return WCSIM_OK;
}

int wcsim_graph_launch(wcsim_graph *graph)
{
    if (!graph) return WCSIM_EINVAL;
    if (graph->plan->capturing) return WCSIM_ESTATE;
    DeviceGuard guard(graph->plan->device);
    if (!guard.ok) return fail_cuda(cudaGetLastError());
    CU_TRY(cudaGraphLaunch(graph->exec, graph->plan->stream));
    graph->plan->launches += graph->launches;
    return WCSIM_OK;
}

int wcsim_graph_destroy(wcsim_graph *graph)
{
    if (!graph) return WCSIM_OK;
    DeviceGuard guard(graph->plan->device);
    cudaStreamSynchronize(graph->plan->stream);
    cudaGraphExecDestroy(graph->exec);
    cudaGraphDestroy(graph->graph);
    graph->plan->live_graphs -= 1;
    delete graph;
    return WCSIM_OK;
}

int wcsim_debug_philox(const unsigned int *dev_ctr, const unsigned int *dev_key, unsigned int *dev_out, long long n,
                       void *cuda_stream)
{
    if (n < 0 || (n > 0 && (!dev_ctr || !dev_key || !dev_out))) return WCSIM_EINVAL;
    CU_TRY(launch_debug_philox(dev_ctr, dev_key, dev_out, n, (cudaStream_t)cuda_stream));
    return WCSIM_OK;
}

int wcsim_digitize(wcsim_plan *plan, float gain, float baseline, int bits, short *dev_adc)
{
    if (!plan || !dev_adc || bits < 1 || bits > 15 || (reinterpret_cast<uintptr_t>(dev_adc) & 7u)) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    if (!guard.ok) return fail_cuda(cudaGetLastError());
    plan->launches += 1;
    CU_TRY(launch_digitize(plan->M, (long long)plan->n_wires * plan->n_ticks, gain, baseline, bits, dev_adc, plan->stream));
    return WCSIM_OK;
}

int wcsim_drift(const float *dev_x, const float *dev_y, const float *dev_z, const float *dev_t, const float *dev_q,
                long long n, const wcsim_drift_params *params, const wcsim_plane_geom *planes, int n_planes,
                const wcsim_depos *out, void *cuda_stream)
{
    if (n < 0 || !params || !planes || !out || n_planes < 1 || n_planes > kMaxDriftPlanes) return WCSIM_EINVAL;
    if (!(params->v_drift > 0.0) || !(params->tick > 0.0) || params->D_L < 0.0 || params->D_T < 0.0) return WCSIM_EINVAL;
    if (n == 0) return WCSIM_OK;
    if (!dev_x || !dev_y || !dev_z || !dev_t || !dev_q) return WCSIM_EINVAL;
    DriftPlanes dp{};
    dp.n = n_planes;
    for (int p = 0; p < n_planes; ++p) {
        if (!(planes[p].pitch > 0.0)) return WCSIM_EINVAL;
        if (!out[p].t0 || !out[p].x0 || !out[p].sigma_t || !out[p].sigma_x || !out[p].q) return WCSIM_EINVAL;
        dp.plane[p] = DriftPlane{planes[p].x_plane, planes[p].cos_theta, planes[p].sin_theta, planes[p].pitch_origin,
                                 planes[p].pitch,
                                 DepoOutputs{const_cast<float *>(out[p].t0), const_cast<float *>(out[p].x0),
                                             const_cast<float *>(out[p].sigma_t), const_cast<float *>(out[p].sigma_x),
                                             const_cast<float *>(out[p].q)}};
    }
    const DriftParams prm{params->v_drift, 2.0 * params->D_L * 1e-6, 2.0 * params->D_T * 1e-6, params->tick,
                          params->t_origin, params->lifetime};
    CU_TRY(launch_drift(DriftInputs{dev_x, dev_y, dev_z, dev_t, dev_q}, n, prm, dp, (cudaStream_t)cuda_stream));
    return WCSIM_OK;
}

int wcsim_debug_erf(const double *host_z, double *host_out, long long n)
{
    if (n < 0 || (n > 0 && (!host_z || !host_out))) return WCSIM_EINVAL;
    erf_table_host(host_z, host_out, n);
    return WCSIM_OK;
}

int wcsim_debug_binomial(const double *dev_N, const double *dev_p, const unsigned int *dev_w, double *dev_k,
                         long long n, void *cuda_stream)
{
    if (n < 0 || (n > 0 && (!dev_N || !dev_p || !dev_w || !dev_k))) return WCSIM_EINVAL;
    CU_TRY(launch_debug_binomial(dev_N, dev_p, dev_w, dev_k, n, false, (cudaStream_t)cuda_stream));
    return WCSIM_OK;
}

int wcsim_debug_normal_draw(const double *dev_N, const double *dev_p, const unsigned int *dev_w, double *dev_k,
                         long long n, void *cuda_stream)
{
    if (n < 0 || (n > 0 && (!dev_N || !dev_p || !dev_w || !dev_k))) return WCSIM_EINVAL;
    CU_TRY(launch_debug_binomial(dev_N, dev_p, dev_w, dev_k, n, true, (cudaStream_t)cuda_stream));
    return WCSIM_OK;
}

int wcsim_debug_fast_normal(const double *dev_N, const double *dev_p, const unsigned int *dev_w, double *dev_k,
                            int *dev_ok, long long n, void *cuda_stream)
{
    if (n < 0 || (n > 0 && (!dev_N || !dev_p || !dev_w || !dev_k || !dev_ok))) return WCSIM_EINVAL;
    CU_TRY(launch_debug_fast_normal(dev_N, dev_p, dev_w, dev_k, dev_ok, n, (cudaStream_t)cuda_stream));
    return WCSIM_OK;
}

int wcsim_debug_z32_scan(unsigned long long first_word, unsigned long long n_words, double *dev_out4, void *cuda_stream)
{
    if (!dev_out4 || first_word + n_words > (1ull << 32)) return WCSIM_EINVAL;
    CU_TRY(launch_debug_z32_scan(first_word, n_words, reinterpret_cast<unsigned long long *>(dev_out4),
                                 (cudaStream_t)cuda_stream));
    return WCSIM_OK;
}

int wcsim_debug_response_spectrum(wcsim_plan *plan, float *host_out)
{
    if (!plan || !host_out) return WCSIM_EINVAL;
    if (!plan->Rhat) return WCSIM_ESTATE; // multi-plane plans keep no Rhat
    DeviceGuard guard(plan->device);
    const int nk = plan->pad_t / 2 + 1;
    CU_TRY(cudaMemcpy2DAsync(host_out, sizeof(float2) * (size_t)nk, plan->Rhat, sizeof(float2) * (size_t)plan->spec_stride,
                             sizeof(float2) * (size_t)nk, (size_t)plan->pad_w, cudaMemcpyDeviceToHost, plan->stream));
    CU_TRY(cudaStreamSynchronize(plan->stream));
    return WCSIM_OK;
}

int wcsim_set_profiling(wcsim_plan *plan, int level)
{
    if (!plan || level < 0 || level > WCSIM_PROFILE_CALLS) return WCSIM_EINVAL;
    plan->profiling = level;
    return WCSIM_OK;
}

int wcsim_get_stage_times(wcsim_plan *plan, double *ms, unsigned long long *calls, int reset)
{
    if (!plan || !ms || !calls) return WCSIM_EINVAL;
    DeviceGuard guard(plan->device);
    const int rc = harvest_spans(plan);
    if (rc) return rc;
    for (int s = 0; s < WCSIM_N_STAGES; ++s) {
        ms[s] = plan->stage_ms[s];
        calls[s] = plan->stage_calls[s];
        if (reset) {
            plan->stage_ms[s] = 0.0;
            plan->stage_calls[s] = 0;
        }
    }
    return WCSIM_OK;
}

int wcsim_get_launch_count(const wcsim_plan *plan, unsigned long long *out)
{
    if (!plan || !out) return WCSIM_EINVAL;
    *out = plan->launches;
    return WCSIM_OK;
}

const char *wcsim_strerror(int status)
{
    switch (status) {
    case WCSIM_OK: return "ok";
    case WCSIM_EINVAL: return "invalid argument";
    case WCSIM_ENOMEM: return "out of host or device memory";
    case WCSIM_ECUDA: return "CUDA runtime or kernel failure (see wcsim_last_cuda_error)";
    case WCSIM_ESTATE: return "call not valid in the plan's current state";
    case WCSIM_ETOOBIG:
        return "grid larger than the built-in scratch of wcsim_raster_scatter_noalloc (n_wires * n_ticks > "
               "WCSIM_NOALLOC_MAX_BINS = 524288); nothing was allocated or enqueued -- use a plan for this size";
    default: return "unknown wcsim status";
    }
}

int wcsim_last_cuda_error(void) { return tls_cuda_error; }

const char *wcsim_version(void) { return "wcsim 0.1 (sm_100a)"; }

} // extern "C"

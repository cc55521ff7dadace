// noalloc.cu -- wcsim_raster_scatter_noalloc: the fixed-point raster + scatter-add (a1-a3) for callers that
// must not allocate device memory.
//
// Who that is: code that runs where cudaMalloc is off the table -- a host framework that hands each plug-in a fixed arena
// and forbids driver allocations once its event loop has started (an allocation takes a device-wide lock and may
// synchronise every stream of the process, which stalls the other plug-ins' work), a real-time data-acquisition thread
// that may not block on the driver, or a process that runs so close to the memory limit that a late cudaMalloc can fail.
// Every other entry point of this library goes through a wcsim_plan, and creating a plan allocates.
//
// What this file does instead: the scratch the kernel needs (the 64-bit fixed-point grid the patches are added into, and
// the kernel's small work-counter block) lives in ONE file-scope device array of a fixed size, which is part of the
// library's image: every GPU that loads libwcsim.so holds those 4 MiB + 256 B from the first CUDA call until the process
// ends, whether or not this entry point is ever used.
//
// The array's name means different things on the two sides of the compiler.  In device code it is the array.  In host
// code it is only a handle for the runtime's symbol table -- not a device address; handing it to a kernel as a pointer
// would make the kernel read host memory (or fault).  So the host side asks the runtime for the device address with
// cudaGetSymbolAddress, once per device and with that device current, and passes THAT to the launchers.
#include "../../include/wcsim.h"
#include "internal.h"

#include <mutex>

using namespace wcsim;

namespace {

constexpr long long kMaxBins = WCSIM_NOALLOC_MAX_BINS;
constexpr int kHeaderWords = 32; // 256 bytes in front of the grid: the kernel's Counters block (32 bytes used)
static_assert(sizeof(Counters) <= kHeaderWords * sizeof(unsigned long long), "counter block does not fit the header");

// words [0, kHeaderWords): Counters;  words [kHeaderWords, kHeaderWords + n_wires * n_ticks): the 2^-24 fixed-point grid
static __device__ __align__(256) unsigned long long g_noalloc_scratch[kHeaderWords + kMaxBins];

struct DeviceSetup {
    bool done = false;
    unsigned long long *scratch = nullptr; // DEVICE address of g_noalloc_scratch on this device
    int sm_count = 0;
};
constexpr int kMaxDevices = 64;
DeviceSetup g_setup[kMaxDevices];
std::mutex g_setup_mutex;

// First call on the current device: resolve the scratch array's device address, read the SM count, upload the erf table
// and set the kernels' shared-memory attributes (raster_configure: synchronises `st` once, allocates nothing).
cudaError_t setup_current_device(cudaStream_t st, DeviceSetup *out)
{
    int dev = -1;
    cudaError_t err = cudaGetDevice(&dev);
    if (err != cudaSuccess) return err;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    DeviceSetup &s = g_setup[dev];
    if (!s.done) {
        void *ptr = nullptr;
        err = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (err != cudaSuccess) return err;
        if (!ptr) return cudaErrorInvalidSymbol;
        int sms = 0;
        err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (err != cudaSuccess) return err;
        err = raster_configure(st);
        if (err != cudaSuccess) return err;
        s.scratch = static_cast<unsigned long long *>(ptr);
        s.sm_count = sms;
        s.done = true;
    }
    *out = s;
    return cudaSuccess;
}

int cuda_status(cudaError_t e)
{
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? WCSIM_ENOMEM : WCSIM_ECUDA;
}

} // namespace

extern "C" int wcsim_raster_scatter_noalloc(int n_wires, int n_ticks, const wcsim_depos *depos, long long n,
                                            unsigned long long depo_id_base, unsigned long long seed, int fluctuate,
                                            float nsigma, float *dev_S, void *cuda_stream)
{
    if (n_wires <= 0 || n_ticks <= 0 || n < 0 || fluctuate < 0 || fluctuate > 2 || !(nsigma > 0.f) || !dev_S)
        return WCSIM_EINVAL;
    const long long n_bins = (long long)n_wires * n_ticks;
    if (n_bins > kMaxBins) return WCSIM_ETOOBIG; // the built-in scratch is all there is: nothing is allocated to make room
    if (n == 0) return WCSIM_OK;
    if (!depos || !depos->t0 || !depos->x0 || !depos->sigma_t || !depos->sigma_x || !depos->q) return WCSIM_EINVAL;

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    DeviceSetup dev;
    cudaError_t err = setup_current_device(st, &dev);
    if (err != cudaSuccess) return cuda_status(err);

    // The array is shared by every call and still holds whatever the last one left (a call that faulted half way leaves
    // charge in the grid and a non-zero work counter), so the part this call uses is zeroed first (a memset: nothing is
    // allocated).
    err = cudaMemsetAsync(dev.scratch, 0, sizeof(unsigned long long) * (size_t)(kHeaderWords + n_bins), st);
    if (err != cudaSuccess) return cuda_status(err);

    Counters *counters = reinterpret_cast<Counters *>(dev.scratch);
    unsigned long long *fix = dev.scratch + kHeaderWords;
    const GridDims g{n_wires, n_ticks};
    const DepoArrays d{depos->t0, depos->x0, depos->sigma_t, depos->sigma_x, depos->q};
    err = launch_raster_fixed(g, d, n, depo_id_base, seed, fluctuate, (double)nsigma, fix, nullptr, counters, dev.sm_count, st);
    if (err != cudaSuccess) return cuda_status(err);
    TileScratch ts{};
    ts.fix = fix;
    err = launch_tile_finalize(g, ts, dev_S, st); // S += fix 2^-24
    if (err != cudaSuccess) return cuda_status(err);
    return WCSIM_OK;
}

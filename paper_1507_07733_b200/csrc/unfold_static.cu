// aera_unfold_batch_static (include/aera_unfold.h): the batch unfolding for callers that cannot allocate device
// memory and cannot hand the library a workspace either.
//
// Who that is: a reconstruction module that runs inside somebody else's process and only ever receives the input
// and output buffers (the host framework owns the device-memory pool and plug-ins are not allowed a cudaMalloc of
// their own, or the pool has already claimed the whole card so a cudaMalloc would simply fail); and a trigger /
// monitoring loop that must not stall: cudaMalloc and cudaFree take a driver-wide lock and synchronise the device,
// which holds up every stream of the process for an unpredictable time.
//
// For them the scratch of the unfolding kernels (the per-event inverse response matrices that minv_kernel writes
// and the unfold kernel reads, plus the transform buffers of the kernel families that need them) lives in ONE
// file-scope __device__ array of AERA_STATIC_SCRATCH_BYTES. It is part of the library image: every GPU on which the
// library's code gets loaded holds these bytes until the process exits, used or not, which is why the size is fixed
// and modest and larger batches are refused rather than served from somewhere else.
//
// Host code must not pass `g_static_scratch` itself to a kernel: on the host that name is only a handle the runtime
// uses to look the array up, not an address on the device. The address is asked for once per device with
// cudaGetSymbolAddress (with that device current) and remembered; device code in this file could name the array
// directly, but the kernels that use it live in other translation units and take the address as their ordinary
// workspace argument.
#include <cstdio>
#include <mutex>

#include "aera_internal.h"

namespace {

// 32 MiB: room for the matrices of 1 000 events at BASELINE configs[1] (20.3 MB) in one call.
constexpr size_t kStaticScratchBytes = (size_t)AERA_STATIC_SCRATCH_BYTES;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];

constexpr int kMaxDevices = 64;
std::mutex g_addr_mu;
void *g_addr[kMaxDevices] = {};   // device address of g_static_scratch on each device, once resolved

// Device address of the array on the CURRENT device. The first call on a device resolves it (this is also what makes
// the runtime load this file's module there, and with it the array's memory); later calls are a table look-up.
cudaError_t static_scratch_address(void **out, int *device)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    *device = dev;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lk(g_addr_mu);
    if (!g_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_addr[dev] = p;
    }
    *out = g_addr[dev];
    return cudaSuccess;
}

} // namespace

extern "C" {

size_t aera_static_scratch_bytes(void) { return kStaticScratchBytes; }

aera_status_t aera_unfold_batch_static(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                                       int n_samples, double fs_hz, const void *traces, const double *dirs,
                                       void *efield, void *peak_amp, int32_t *peak_idx, void *cuda_stream)
{
    using namespace aera;
    if (!pattern) return report_error(AERA_ERR_INVALID_ARG, "pattern is NULL");
    if (n_events < 0) return report_error(AERA_ERR_INVALID_ARG, "n_events is negative");
    if (n_events == 0) return AERA_OK;
    // the plan of a new (n_samples, fs_hz) pair is a cudaMalloc + upload: that belongs to set-up, not to this call
    if (!plan_is_cached(pattern, n_samples, fs_hz))
        return report_error(AERA_ERR_INVALID_ARG,
                            "aera_unfold_batch_static allocates nothing, and this pattern has no plan for this (n_samples, fs_hz) yet: "
                            "call aera_pattern_prepare(pattern, n_samples, fs_hz, stream) once at set-up");
    const size_t need = aera_workspace_bytes(AERA_OP_UNFOLD, pattern, dtype, n_events, n_stations, n_samples, fs_hz);
    if (need == 0) return AERA_ERR_INVALID_ARG;                       // aera_workspace_bytes has set the message
    if (need > kStaticScratchBytes) {
        char msg[320];
        snprintf(msg, sizeof(msg),
                 "this batch needs %zu bytes of scratch but the built-in scratch array holds %zu (AERA_STATIC_SCRATCH_BYTES): "
                 "split the events over several calls, or use aera_unfold_batch with a workspace of your own",
                 need, kStaticScratchBytes);
        return report_error(AERA_ERR_WORKSPACE, msg);
    }
    void *scratch = nullptr;
    int dev = -1;
    cudaError_t e = static_scratch_address(&scratch, &dev);
    if (e != cudaSuccess) {
        (void)cudaGetLastError();
        char msg[200];
        snprintf(msg, sizeof(msg), "cudaGetSymbolAddress of the built-in scratch array on device %d: %s", dev, cudaGetErrorString(e));
        return report_error(AERA_ERR_CUDA, msg);
    }
    // Nothing in the scratch has to start at zero: every entry the unfold kernels read (zero pads of the matrix planes
    // included) is written by minv_kernel or by the unfold kernel itself earlier in the same call, so what the previous
    // call left behind is never seen. From here on this is the ordinary path with the array as its workspace.
    return aera_unfold_batch(pattern, dtype, n_events, n_stations, n_samples, fs_hz, traces, dirs, efield, peak_amp, peak_idx,
                             scratch, kStaticScratchBytes, cuda_stream);
}

} // extern "C"

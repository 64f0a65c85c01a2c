// Measured ALU peaks of the device the library runs on: the denominators of the "alu" roofline that
// bench.py reports for the FP32-pipe-bound scan mode (BASELINE north_star: "FP32/FP64 pipe utilisation
// for the scan mode") and of the FP32 / FP64 co-limiter figures in DESIGN.md section 5.
//
// Each kernel is a register-only chain of independent fused multiply-adds, 8 accumulators per thread,
// unrolled 32x, one CTA per SM x `ctas_per_sm`, so the only limiter is the issue rate of the pipe:
//   kind 0  fma.rn.f32x2 (SASS FFMA2): two fp32 FMAs per lane per instruction (the warp kernels' form)
//   kind 1  fma.rn.f32   (SASS FFMA)
//   kind 2  fma.rn.f64   (SASS DFMA)
// Result: lane-FMAs per second over the whole device (x 2 = FLOP/s).
#include "aera_internal.h"
#include "fft32.cuh"

namespace aera {
namespace {

template <int KIND>
__global__ void __launch_bounds__(1024, 1) alu_peak_kernel(double *out, int iters, float a, float b)
{
    if constexpr (KIND == 0) {
        F2 x[8];
        const F2 pa = LaneF32x2::pack(a, a), pb = LaneF32x2::pack(b, b);
        for (int i = 0; i < 8; ++i) x[i] = LaneF32x2::pack(threadIdx.x * 1e-3f + i, i * 0.5f);
#pragma unroll 1
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < 32; ++u)
#pragma unroll
                for (int i = 0; i < 8; ++i) x[i] = LaneF32x2::fma(x[i], pa, pb);
        }
        float s = 0.f;
        for (int i = 0; i < 8; ++i) { float lo, hi; LaneF32x2::unpack(x[i], lo, hi); s += lo + hi; }
        out[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = s;
    } else if constexpr (KIND == 1) {
        float x[8];
        for (int i = 0; i < 8; ++i) x[i] = threadIdx.x * 1e-3f + i;
#pragma unroll 1
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < 32; ++u)
#pragma unroll
                for (int i = 0; i < 8; ++i) x[i] = fmaf(x[i], a, b);
        }
        float s = 0.f;
        for (int i = 0; i < 8; ++i) s += x[i];
        out[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = s;
    } else {
        double x[8];
        const double da = a, db = b;
        for (int i = 0; i < 8; ++i) x[i] = threadIdx.x * 1e-3 + i;
#pragma unroll 1
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int u = 0; u < 32; ++u)
#pragma unroll
                for (int i = 0; i < 8; ++i) x[i] = fma(x[i], da, db);
        }
        double s = 0.0;
        for (int i = 0; i < 8; ++i) s += x[i];
        out[blockIdx.x * (size_t)blockDim.x + threadIdx.x] = s;
    }
}

template <int KIND>
cudaError_t run_kind(int sms, int warps, int iters, double *d_out, double *lane_fma_per_s)
{
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    e = cudaEventCreate(&e1);
    if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
    double best = 0.0;
    alu_peak_kernel<KIND><<<sms, warps * 32>>>(d_out, 16, 1.0000001f, 1e-9f);          // warm-up
    for (int rep = 0; rep < 3 && e == cudaSuccess; ++rep) {
        cudaEventRecord(e0);
        alu_peak_kernel<KIND><<<sms, warps * 32>>>(d_out, iters, 1.0000001f, 1e-9f);
        cudaEventRecord(e1);
        e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        const double fmas = (double)sms * warps * 32 * (double)iters * 256.0 * (KIND == 0 ? 2.0 : 1.0);
        if (e == cudaSuccess && ms > 0.f && fmas / (ms * 1e-3) > best) best = fmas / (ms * 1e-3);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e == cudaSuccess) e = cudaGetLastError();
    *lane_fma_per_s = best;
    return e;
}

} // namespace

cudaError_t measure_alu_peak(int kind, int warps_per_sm, double *lane_fma_per_s, int *sm_count, int *sm_clock_khz)
{
    int dev = 0, sms = 0, khz = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
    if (e != cudaSuccess) return e;
    double *d_out = nullptr;
    e = cudaMalloc((void **)&d_out, (size_t)sms * 1024 * sizeof(double));
    if (e != cudaSuccess) return e;
    const int iters = 1000;
    if (kind == 0) e = run_kind<0>(sms, warps_per_sm, iters, d_out, lane_fma_per_s);
    else if (kind == 1) e = run_kind<1>(sms, warps_per_sm, iters, d_out, lane_fma_per_s);
    else e = run_kind<2>(sms, warps_per_sm, iters, d_out, lane_fma_per_s);
    cudaFree(d_out);
    count_launches(4);
    *sm_count = sms; *sm_clock_khz = khz;
    return e;
}

} // namespace aera

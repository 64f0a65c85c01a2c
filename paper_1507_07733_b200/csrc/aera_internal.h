// Internal declarations shared by the translation units of libaera_unfold.so.
// Nothing here is part of the C ABI (include/aera_unfold.h) and nothing here is shared with oracle/.
#pragma once
#include <atomic>
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>

#include "../../include/aera_unfold.h"

namespace aera {

template <typename T> struct cx { T re, im; };

// Geometry of the repacked table [n_z][n_a][n_f][4] (4 = channel*2 + pol).
struct TableGeom {
    int n_z, n_a, n_f, periodic;
    double z0, dz, a0, da;
};

// Everything a kernel needs to know about one (pattern, N, fs) combination. Device pointers are
// owned by the pattern handle (built on first use, see api.cu).
struct PlanDev {
    int N, logN;
    int k_lo, k_hi, K;
    const int *bin_if;      // [K] lower frequency node of bin k_lo+j
    const double *bin_tf;   // [K] weight of the upper node
    const double *bin_w;    // [K] optional pre-filter weight per in-band bin (NULL = none), folded into Minv
    const void *tw;         // [N/2] cx<T>: W_N^m = exp(-2 pi i m / N), m < N/2 (generic kernel)
    const void *tw1024;     // [1024] cx<T>: W_1024^m (warp kernels: 32x32 inter-pass twiddles)
    const void *twN;        // [N] cx<T>: W_N^m, m < N (real-FFT split / polyphase twiddles)
    int U, logM;            // spectral up-sampling factor (1 = none) and log2(U N)
    const void *twU;        // [U N / 2] cx<T>: W_{UN}^m (generic kernel's inverse transform on the fine grid; = tw when U = 1)
};

// Variations of the batch unfolding beyond one table / real-typed traces / the input sampling grid
// (aera_unfold_batch_multi, aera_unfold_batch_i16, aera_unfold_batch_upsampled).
struct UnfoldExt {
    const int32_t *pattern_id = nullptr; // device [n_stations]: antenna type of each station (nullptr: one table)
    size_t minv_pattern_stride = 0;      // complex elements between the Minv slabs of consecutive tables (= n_events * per-event size)
    int input_i16 = 0;                   // traces are int16 ADC counts (the counts-to-volts factors are folded into Minv)
};

void count_launches(unsigned n);
int kernel_variant();

// Optional per-kernel CUDA-event timing (aera_profile_enable / aera_profile_read in the C ABI).
enum KernelId { KID_REPACK = 0, KID_MINV = 1, KID_UNFOLD = 2, KID_SCAN_FWD = 3, KID_SCAN_INV = 4, KID_TIMING = 5, KID_PLANEFIT = 6, KID_COUNT = 7 };
void prof_begin(int kid, cudaStream_t s); // no-ops unless profiling is enabled
void prof_end(int kid, cudaStream_t s);
struct ProfScope {
    int kid; cudaStream_t s;
    ProfScope(int k, cudaStream_t st) : kid(k), s(st) { prof_begin(kid, s); }
    ~ProfScope() { prof_end(kid, s); }
};

// Function attributes, device limits and device properties belong to ONE device: what the library remembers about them
// is kept per device ordinal, so a process may use the library on several GPUs (one after the other or from several
// threads, each with its own current device).
constexpr int kMaxDevices = 64;
// slot of the current device in such a table, or -1 (unknown / beyond the table: nothing is remembered for it)
inline int device_slot()
{
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return -1; }
    return (dev >= 0 && dev < kMaxDevices) ? dev : -1;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize raised once per kernel and device (and again only if a call needs more),
// not on every launch: the table is a static of the call site, one per kernel instantiation.
#define AERA_ENSURE_DYN_SMEM(kern, bytes)                                                                   \
    do {                                                                                                    \
        static std::atomic<size_t> aera_cur_smem[::aera::kMaxDevices];                                      \
        const int aera_slot = ::aera::device_slot();                                                        \
        if (aera_slot < 0 || (size_t)(bytes) > aera_cur_smem[aera_slot].load(std::memory_order_acquire)) {  \
            cudaError_t aera_e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bytes)); \
            if (aera_e != cudaSuccess) return aera_e;                                                       \
            if (aera_slot >= 0) aera_cur_smem[aera_slot].store((size_t)(bytes), std::memory_order_release); \
        }                                                                                                   \
    } while (0)

// ---- peaks.cu: measured ALU issue peaks (aera_measure_alu_peak)
cudaError_t measure_alu_peak(int kind, int warps_per_sm, double *lane_fma_per_s, int *sm_count, int *sm_clock_khz);
// number of SMs of the current device (cached per device; api.cu)
int sm_count();
// records the kernel family a call dispatched to (aera_last_kernel)
void note_kernel(const char *name);

// ---- api.cu hooks of unfold_static.cu (aera_unfold_batch_static)
// sets the thread's aera_last_error() message and returns st
aera_status_t report_error(aera_status_t st, const char *msg);
// whether the plan of (n_samples, fs_hz), up-sampling 1, is already built: a look-up, never a build
bool plan_is_cached(const aera_pattern_t *pattern, int n_samples, double fs_hz);

// ---- pattern.cu
cudaError_t launch_repack(int dtype, const void *src, void *dst, int n_z, int n_a, int n_f, cudaStream_t s);
// Minv[d][j][4] = scale * H(theta_d, phi_d, f_{k_lo+j})^-1.
//   MINV_ROWS   : complex entries (theta<-V0, theta<-V1, phi<-V0, phi<-V1)            (generic kernels)
//   MINV_PACKED : per direction two planes A[K], B[K] of 4 reals: A = {t0.re, p0.re, t0.im, p0.im},
//                 B = {t1.re, p1.re, t1.im, p1.im}                                     (warp kernels)
//   MINV_Q4     : per direction 16 planes [q = k & 3][entry 0..3 as in MINV_ROWS][C] complex, column
//                 (k >> 2) - (k_lo >> 2), C = (k_hi >> 2) - (k_lo >> 2) + 1; slots of bins outside the
//                 band are never written or used                                       (team kernel, teams of 4 warps)
//   MINV_Q2, MINV_Q1, MINV_Q8, MINV_Q16 : the same with q = k mod 2 / 1 / 8 / 16 (4 tw planes)  (teams of 2 / 1 / 8 / 16 warps)
//   MINV_Q32    : per direction 64 float4 planes [q = k & 31][A | B as in MINV_PACKED][C], column
//                 (k >> 5) - (k_lo >> 5), C = (k_hi >> 5) - (k_lo >> 5) + 1              (long-trace kernel)
//   MINV_PACKED_PAD : MINV_PACKED with 32 zero entries before and after each plane (planes of K + 64 entries, bin j at
//                 index j + 32): a warp kernel whose edge rows reach up to 31 bins beyond the band multiplies by zero
//                 there instead of clamping the index and selecting                       (batch warp kernel)
enum MinvLayout { MINV_ROWS = 0, MINV_PACKED = 1, MINV_Q4 = 2, MINV_Q32 = 3, MINV_PACKED_PAD = 4, MINV_Q2 = 5, MINV_Q1 = 6, MINV_Q8 = 7, MINV_Q16 = 8 };
constexpr int kMinvPad = 32;
// complex elements per direction in the MINV_Q4 / Q2 / Q1 layouts, tw = 4 / 2 / 1 (<= 4 K + 8 tw)
__host__ __device__ inline size_t minv_qt_stride(int tw, int k_lo, int k_hi) { return (size_t)4 * tw * ((k_hi / tw) - (k_lo / tw) + 1); }
cudaError_t launch_minv(int dtype, const void *table, const TableGeom &g, const PlanDev &p,
                        const double *dirs, long n_dirs, void *minv, int layout, double scale, cudaStream_t s,
                        int forward = 0 /* 1: scale * H (forward model) instead of scale * H^-1 */,
                        double chan_scale0 = 1.0, double chan_scale1 = 1.0 /* per-channel input scale folded into the columns */);
size_t minv_smem_bytes(int dtype, int n_f);
// out[i] = pattern_id[i] clamped to 0 .. n_patterns-1 (device to device; aera_unfold_batch_multi)
cudaError_t launch_clamp_pattern_id(const int32_t *pattern_id, int32_t *out, int n_stations, int n_patterns, cudaStream_t s);

// ---- unfold_generic.cu
size_t generic_scratch_bytes(int dtype, int N, long n_units, int upsample = 1);   // per-call global transform buffers (0 if smem-resident)
cudaError_t launch_unfold_generic(int dtype, const PlanDev &p, long n_events, int n_stations,
                                  const void *traces, void *efield, void *amp, int32_t *idx,
                                  const void *minv, void *scratch, cudaStream_t s, const UnfoldExt &x = UnfoldExt());
size_t generic_scan_spectra_bytes(int dtype, int K, int n_stations);
cudaError_t launch_scan_generic(int dtype, const PlanDev &p, int n_stations, const void *traces,
                                long n_dirs, const void *minv, void *amp, int32_t *idx,
                                void *spectra, void *scratch, cudaStream_t s);

// ---- unfold_w32.cu: warp-per-station kernel for N = 2048 fp32 with the band below N/2
bool w32_supported(int dtype, const PlanDev &p);
// spectra / spec_mode: 1 = also store the direction-independent band spectra 2 V_c, 2 = start from them (no trace
// read, no forward transform); w32_spectra_bytes() = 0 when the band geometry has no such instantiation
size_t w32_spectra_bytes(const PlanDev &p, long n_units);
cudaError_t launch_unfold_w32(const PlanDev &p, long n_events, int n_stations, const void *traces, void *efield,
                              void *amp, int32_t *idx, const void *minv, cudaStream_t s, void *spectra = nullptr, int spec_mode = 0,
                              const UnfoldExt &x = UnfoldExt());

// ---- unfold_t4k.cu: team-per-station kernel, N = 1024 x (warps of a team): 4096 fp64 (configs[3]) / fp32, 2048 fp64, 1024 fp64 / fp32
bool t4k_supported(int dtype, const PlanDev &p);
int t4k_team_warps(int dtype, const PlanDev &p);
// (the fp32 and the int16-input instantiations live in their own translation units, unfold_t4k_f32.cu / unfold_t4k_i16.cu)
cudaError_t launch_unfold_t4k_i16(const PlanDev &p, long n_units, int n_stations, const void *traces, void *efield, void *amp,
                                  int32_t *idx, const void *minv, cudaStream_t s, const UnfoldExt &x);
cudaError_t launch_unfold_t4k_f32(const PlanDev &p, long n_units, int n_stations, const void *traces, void *efield, void *amp,
                                  int32_t *idx, const void *minv, cudaStream_t s, const UnfoldExt &x);   // 4, 2, 1, or 0 when the kernel does not cover (dtype, N, band)
cudaError_t launch_unfold_t4k(int dtype, const PlanDev &p, long n_events, int n_stations, const void *traces, void *efield,
                                  void *amp, int32_t *idx, const void *minv, cudaStream_t s, const UnfoldExt &x = UnfoldExt());

// ---- unfold_long_f32.cu: multi-pass kernel for N = 65536 fp32 through an L2-resident scratch (configs[4])
bool long_f32_supported(int dtype, const PlanDev &p);
size_t long_f32_scratch_bytes(const PlanDev &p);
long set_long_persist_mb(long mb);   // aera_set_long_trace_l2_persist; returns the previous request
cudaError_t launch_unfold_long_f32(const PlanDev &p, long n_events, int n_stations, const void *traces, void *efield,
                                   void *amp, int32_t *idx, const void *minv, void *scratch, cudaStream_t s,
                                   const UnfoldExt &x = UnfoldExt());

// ---- loop.cu: the two small steps that close the reconstruction loop on the device
cudaError_t launch_timing(int dtype, const void *traces, long n_units, int N, int32_t *idx0, void *w0, cudaStream_t s);
cudaError_t launch_planefit(int dtype, const double *pos, const int32_t *idx, const void *w, int square_w, long n_events,
                            int n_stations, double fs, double *dirs, cudaStream_t s);

cudaError_t launch_convergence(const double *dirs_hist, int n_iter, long n_events, double tol_deg, int32_t *conv_iter, cudaStream_t s);

// ---- scan_w32.cu: direction scan for N = 2048 fp32, band rows 10..28 (configs[2])
bool scan_w32_supported(int dtype, const PlanDev &p);
size_t scan_w32_spectra_bytes(int n_stations);
cudaError_t launch_scan_w32(const PlanDev &p, int n_stations, const void *traces, long n_dirs, const void *minv,
                            void *amp, int32_t *idx, void *spectra, cudaStream_t s);

} // namespace aera

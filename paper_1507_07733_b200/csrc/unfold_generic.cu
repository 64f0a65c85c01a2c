// Generic unfolding kernels: any power-of-two N in [64, 65536], fp32 or fp64.
//
// This is the library's reference-quality CUDA path: one CTA per station, in-place radix-2
// transforms on three complex buffers (forward spectrum, Z_theta, Z_phi) that live in shared
// memory when they fit (3*N*sizeof(complex) <= 192 KB) and otherwise in a per-CTA slice of the
// caller's workspace (L2-resident).  It covers every size the specialised warp kernels
// (unfold_w32.cu) do not, and tests run it against them.  Steps per station:
//   a1 load v0 + i v1 (bit-reversed)           a2 forward FFT (two real transforms for one)
//   a4 E = Minv V on the in-band bins           a5 two inverse FFTs of the one-sided spectra
//   a6 e_p = Re z_p, env^2 = |z_theta|^2+|z_phi|^2, max / lowest argmax
// (a3, the pattern evaluation, is pattern.cu's minv_kernel, once per event.)
#include "aera_internal.h"

namespace aera {

namespace {

constexpr int kThreads = 256;
constexpr size_t kSmemBudget = 192 * 1024;

template <typename T>
__device__ __forceinline__ cx<T> cmul(cx<T> a, cx<T> b)
{
    cx<T> r;
    r.re = a.re * b.re - a.im * b.im;
    r.im = a.re * b.im + a.im * b.re;
    return r;
}

// In-place decimation-in-time FFT of NBUF buffers of N points whose inputs are already in bit-reversed order.
// tw[m] = exp(-2 pi i m / N), m < N/2; inverse uses the conjugate. Three radix-2 stages are fused into one
// radix-8 pass per trip through shared memory (each thread holds the 8 points i0 + t 2^s, t = 0..7, of a group in
// registers), preceded by one radix-2 or radix-4 pass when log2 N is not a multiple of 3: a third of the
// barriers and of the shared-memory traffic of the stage-by-stage form.
template <typename T, bool INVERSE>
__device__ __forceinline__ void bfly(cx<T> &a, cx<T> &b, cx<T> w)
{
    if (INVERSE) w.im = -w.im;
    const cx<T> t = cmul(w, b);
    b.re = a.re - t.re; b.im = a.im - t.im;
    a.re = a.re + t.re; a.im = a.im + t.im;
}
// LOG_R fused stages starting at stage s on the group g of buffer b
template <typename T, bool INVERSE, int LOG_R>
__device__ __forceinline__ void radix_group(cx<T> *b, int g, int s, int N, const cx<T> *__restrict__ tw)
{
    constexpr int R = 1 << LOG_R;
    const int pos = g & ((1 << s) - 1);
    const int i0 = ((g >> s) << (s + LOG_R)) + pos;
    cx<T> x[R];
#pragma unroll
    for (int t = 0; t < R; ++t) x[t] = b[i0 + (t << s)];
#pragma unroll
    for (int l = 0; l < LOG_R; ++l) {                  // stage s + l pairs local t and t + 2^l
        const int tstride = (N >> 1) >> (s + l);
#pragma unroll
        for (int t = 0; t < R; ++t) {
            if (t & (1 << l)) continue;
            const int p = pos + ((t & ((1 << l) - 1)) << s);   // position of the pair inside its 2^(s+l+1) block
            bfly<T, INVERSE>(x[t], x[t + (1 << l)], tw[p * tstride]);
        }
    }
#pragma unroll
    for (int t = 0; t < R; ++t) b[i0 + (t << s)] = x[t];
}
template <typename T, bool INVERSE, int NBUF, int LOG_R>
__device__ __forceinline__ void radix_pass(cx<T> *b0, cx<T> *b1, int s, int N, const cx<T> *__restrict__ tw)
{
    for (int g = threadIdx.x; g < (N >> LOG_R); g += blockDim.x) {
        radix_group<T, INVERSE, LOG_R>(b0, g, s, N, tw);
        if (NBUF == 2) radix_group<T, INVERSE, LOG_R>(b1, g, s, N, tw);
    }
    __syncthreads();
}
template <typename T, bool INVERSE, int NBUF>
__device__ void cta_fft(cx<T> *b0, cx<T> *b1, int N, int logN, const cx<T> *__restrict__ tw)
{
    int s = 0;
    const int r = logN % 3;
    if (r == 1) { radix_pass<T, INVERSE, NBUF, 1>(b0, b1, 0, N, tw); s = 1; }
    else if (r == 2) { radix_pass<T, INVERSE, NBUF, 2>(b0, b1, 0, N, tw); s = 2; }
    for (; s < logN; s += 3) radix_pass<T, INVERSE, NBUF, 3>(b0, b1, s, N, tw);
}

// (value, index) max with lowest index on ties; every reduction stage uses the same rule.
template <typename T>
__device__ __forceinline__ void argmax_combine(T &v, int &i, T ov, int oi)
{
    if (ov > v || (ov == v && oi < i)) { v = ov; i = oi; }
}

template <typename T>
__device__ void cta_argmax(T v, int i, T *amp_out, int32_t *idx_out)
{
    __shared__ T sv[32];
    __shared__ int si[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        T ov = __shfl_xor_sync(0xffffffffu, v, o);
        int oi = __shfl_xor_sync(0xffffffffu, i, o);
        argmax_combine(v, i, ov, oi);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sv[warp] = v; si[warp] = i; }
    __syncthreads();
    if (warp == 0) {
        const int nw = blockDim.x >> 5;
        v = lane < nw ? sv[lane] : (T)-1;
        i = lane < nw ? si[lane] : 0x7fffffff;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            T ov = __shfl_xor_sync(0xffffffffu, v, o);
            int oi = __shfl_xor_sync(0xffffffffu, i, o);
            argmax_combine(v, i, ov, oi);
        }
        if (lane == 0) { *amp_out = sqrt(v); *idx_out = i; }
    }
    __syncthreads();
}

template <typename T>
__device__ __forceinline__ void zero_buffers(cx<T> *B, cx<T> *C, int N)
{
    for (int n = threadIdx.x; n < N; n += blockDim.x) {
        B[n].re = 0; B[n].im = 0; C[n].re = 0; C[n].im = 0;
    }
}

// a5 + a6 on buffers B (theta) and C (phi) holding the bit-reversed one-sided spectra.
// With spectral up-sampling (p.U > 1) the buffers hold M = U N points and the transform is the inverse DFT of
// length M of the same (zero-padded) spectrum: z[n] on a grid U times finer (aera_unfold_batch_upsampled).
template <typename T>
__device__ void inverse_and_peak(cx<T> *B, cx<T> *C, const PlanDev &p, T *ef, T *amp, int32_t *idx)
{
    const int N = p.N * p.U;
    cta_fft<T, true, 2>(B, C, N, p.logM, (const cx<T> *)p.twU);
    T best = (T)-1; int bi = 0x7fffffff;
    for (int n = threadIdx.x; n < N; n += blockDim.x) {
        cx<T> zt = B[n], zp = C[n];
        if (ef) { ef[n] = zt.re; ef[N + n] = zp.re; }
        T e2 = zt.re * zt.re + zt.im * zt.im + zp.re * zp.re + zp.im * zp.im;
        argmax_combine(best, bi, e2, n);
    }
    cta_argmax<T>(best, bi, amp, idx);
}

// IN = T, or int16_t for ADC-count input (the counts-to-volts factors are in Minv)
template <typename T, typename IN>
__device__ void forward_spectrum(cx<T> *A, const PlanDev &p, const IN *v)
{
    const int N = p.N, sh = 32 - p.logN;
    for (int n = threadIdx.x; n < N; n += blockDim.x) {
        const int r = (int)(__brev((unsigned)n) >> sh);
        A[r].re = (T)v[n]; A[r].im = (T)v[N + n];
    }
    __syncthreads();
    cta_fft<T, false, 1>(A, nullptr, N, p.logN, (const cx<T> *)p.tw);
}

// C[k] = V0[k] + i V1[k], conj C[N-k] = V0[k] - i V1[k]  (v0, v1 real)
template <typename T>
__device__ __forceinline__ void split_channels(cx<T> c, cx<T> m, cx<T> &v0, cx<T> &v1)
{
    v0.re = (T)0.5 * (c.re + m.re); v0.im = (T)0.5 * (c.im - m.im);
    v1.re = (T)0.5 * (c.im + m.im); v1.im = (T)-0.5 * (c.re - m.re);
}

template <typename T>
__device__ __forceinline__ void apply_minv(const cx<T> *__restrict__ M, cx<T> v0, cx<T> v1, cx<T> &et, cx<T> &ep)
{
    cx<T> a = cmul(M[0], v0), b = cmul(M[1], v1);
    et.re = a.re + b.re; et.im = a.im + b.im;
    a = cmul(M[2], v0); b = cmul(M[3], v1);
    ep.re = a.re + b.re; ep.im = a.im + b.im;
}

template <typename T, bool SMEM, typename IN>
__global__ void __launch_bounds__(kThreads)
unfold_generic_kernel(PlanDev p, long n_units, int n_stations, const IN *__restrict__ traces, T *efield,
                      T *__restrict__ amp, int32_t *__restrict__ idx, const cx<T> *__restrict__ minv,
                      cx<T> *scratch, const int32_t *__restrict__ pattern_id, size_t minv_pattern_stride)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = p.N, M_ = p.N * p.U, shM = 32 - p.logM;   // transform sizes: forward N, inverse M_ = U N
    cx<T> *A = SMEM ? reinterpret_cast<cx<T> *>(smem_raw) : scratch + (size_t)blockIdx.x * (N + 2 * (size_t)M_);
    cx<T> *B = A + N, *C = B + M_;

    for (long u = blockIdx.x; u < n_units; u += gridDim.x) {
        const long ev = u / n_stations;
        zero_buffers(B, C, M_);
        forward_spectrum<T, IN>(A, p, traces + (size_t)u * 2 * N); // ends with __syncthreads
        // one Minv per (event, antenna type of the station) when several tables are resident
        const cx<T> *M = minv + (pattern_id ? (size_t)pattern_id[u - ev * n_stations] * minv_pattern_stride : 0) + (size_t)ev * p.K * 4;
        for (int j = threadIdx.x; j < p.K; j += blockDim.x) {
            const int k = p.k_lo + j;
            cx<T> v0, v1, et, ep;
            split_channels(A[k], A[N - k], v0, v1);
            apply_minv(M + 4 * j, v0, v1, et, ep);
            const int r = (int)(__brev((unsigned)k) >> shM);    // bin k of the length-M_ spectrum (zero-padded above the band)
            B[r] = et; C[r] = ep;
        }
        __syncthreads();
        inverse_and_peak<T>(B, C, p, efield ? efield + (size_t)u * 2 * M_ : nullptr, amp + u, idx + u);
    }
}

// Scan, kernel A: forward transform once per station, in-band spectra to the workspace [S][2][K].
template <typename T, bool SMEM>
__global__ void __launch_bounds__(kThreads)
scan_forward_generic_kernel(PlanDev p, int n_stations, const T *__restrict__ traces, cx<T> *__restrict__ spectra,
                            cx<T> *scratch)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = p.N;
    cx<T> *A = SMEM ? reinterpret_cast<cx<T> *>(smem_raw) : scratch + (size_t)blockIdx.x * 3 * N;
    for (int s = blockIdx.x; s < n_stations; s += gridDim.x) {
        forward_spectrum<T, T>(A, p, traces + (size_t)s * 2 * N);
        for (int j = threadIdx.x; j < p.K; j += blockDim.x) {
            const int k = p.k_lo + j;
            cx<T> v0, v1;
            split_channels(A[k], A[N - k], v0, v1);
            spectra[((size_t)s * 2 + 0) * p.K + j] = v0;
            spectra[((size_t)s * 2 + 1) * p.K + j] = v1;
        }
        __syncthreads();
    }
}

// Scan, kernel B: one CTA per (direction, station) pair.
template <typename T, bool SMEM>
__global__ void __launch_bounds__(kThreads)
scan_inverse_generic_kernel(PlanDev p, int n_stations, long n_pairs, const cx<T> *__restrict__ spectra,
                            const cx<T> *__restrict__ minv, T *__restrict__ amp, int32_t *__restrict__ idx,
                            cx<T> *scratch)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int N = p.N, sh = 32 - p.logN;
    cx<T> *A = SMEM ? reinterpret_cast<cx<T> *>(smem_raw) : scratch + (size_t)blockIdx.x * 3 * N;
    cx<T> *B = A + N, *C = B + N;
    for (long pr = blockIdx.x; pr < n_pairs; pr += gridDim.x) {
        const long d = pr / n_stations;
        const int s = (int)(pr % n_stations);
        zero_buffers(B, C, N);
        __syncthreads();
        const cx<T> *M = minv + (size_t)d * p.K * 4;
        for (int j = threadIdx.x; j < p.K; j += blockDim.x) {
            cx<T> et, ep;
            apply_minv(M + 4 * j, spectra[((size_t)s * 2 + 0) * p.K + j], spectra[((size_t)s * 2 + 1) * p.K + j], et, ep);
            const int r = (int)(__brev((unsigned)(p.k_lo + j)) >> sh);
            B[r] = et; C[r] = ep;
        }
        __syncthreads();
        inverse_and_peak<T>(B, C, p, (T *)nullptr, amp + pr, idx + pr);
    }
}

size_t elem_bytes(int dtype) { return dtype == AERA_F32 ? sizeof(cx<float>) : sizeof(cx<double>); }
bool fits_smem(int dtype, int N, int U = 1) { return ((size_t)N + 2 * (size_t)N * U) * elem_bytes(dtype) <= kSmemBudget; }
int generic_threads(int N) { const int t = N / 4; return t < 32 ? 32 : (t > kThreads ? kThreads : t); }
long generic_grid(long n_units) { return n_units < (long)sm_count() * 4 ? n_units : (long)sm_count() * 4; }

template <typename K>
cudaError_t set_smem(K kernel, size_t bytes)
{
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

template <typename T, typename IN>
cudaError_t launch_unfold_t(int dtype, const PlanDev &p, long n_units, int n_stations, const void *traces, void *efield,
                            void *amp, int32_t *idx, const void *minv, void *scratch, cudaStream_t s, const UnfoldExt &x)
{
    ProfScope prof(KID_UNFOLD, s);
    // short traces: fewer threads per CTA and more CTAs per SM (256 threads on 64 points leave three quarters of them
    // idle at every barrier; measured fp32 N = 64 / 128 / 256 / 512: 182 / 307 / 498 / 502 -> 551 / 601 / 651 / 553 GB/s)
    const int threads = generic_threads(p.N);
    const long per_sm = 2048 / threads > 32 ? 32 : 2048 / threads;
    const long small_grid = n_units < (long)sm_count() * per_sm ? n_units : (long)sm_count() * per_sm;
    // the global-scratch path has one slice per CTA of generic_grid (generic_scratch_bytes sizes it so): it must never
    // run on the larger small_grid, which a short trace with a large up-sampling factor (N + 2 N U beyond shared
    // memory, e.g. fp32 N = 512, U = 32) would otherwise select
    const bool smem_path = fits_smem(dtype, p.N, p.U);
    const long grid = (smem_path && threads < kThreads) ? small_grid : generic_grid(n_units);
    if (smem_path) {
        size_t smem = ((size_t)p.N + 2 * (size_t)p.N * p.U) * sizeof(cx<T>);
        cudaError_t e = set_smem(unfold_generic_kernel<T, true, IN>, smem);
        if (e != cudaSuccess) return e;
        unfold_generic_kernel<T, true, IN><<<(unsigned)grid, threads, smem, s>>>(
            p, n_units, n_stations, (const IN *)traces, (T *)efield, (T *)amp, idx, (const cx<T> *)minv, nullptr,
            x.pattern_id, x.minv_pattern_stride);
    } else {
        unfold_generic_kernel<T, false, IN><<<(unsigned)grid, kThreads, 0, s>>>(
            p, n_units, n_stations, (const IN *)traces, (T *)efield, (T *)amp, idx, (const cx<T> *)minv, (cx<T> *)scratch,
            x.pattern_id, x.minv_pattern_stride);
    }
    count_launches(1);
    return cudaGetLastError();
}

template <typename T>
cudaError_t launch_scan_t(int dtype, const PlanDev &p, int n_stations, const void *traces, long n_dirs, const void *minv,
                          void *amp, int32_t *idx, void *spectra, void *scratch, cudaStream_t s)
{
    const long n_pairs = n_dirs * (long)n_stations;
    const long gridA = generic_grid(n_stations), gridB = generic_grid(n_pairs);
    if (fits_smem(dtype, p.N)) {
        size_t smem = (size_t)3 * p.N * sizeof(cx<T>);
        cudaError_t e = set_smem(scan_forward_generic_kernel<T, true>, smem);
        if (e != cudaSuccess) return e;
        e = set_smem(scan_inverse_generic_kernel<T, true>, smem);
        if (e != cudaSuccess) return e;
        {
            ProfScope prof(KID_SCAN_FWD, s);
            scan_forward_generic_kernel<T, true><<<(unsigned)gridA, kThreads, smem, s>>>(
                p, n_stations, (const T *)traces, (cx<T> *)spectra, nullptr);
        }
        ProfScope prof(KID_SCAN_INV, s);
        scan_inverse_generic_kernel<T, true><<<(unsigned)gridB, kThreads, smem, s>>>(
            p, n_stations, n_pairs, (const cx<T> *)spectra, (const cx<T> *)minv, (T *)amp, idx, nullptr);
    } else {
        {
            ProfScope prof(KID_SCAN_FWD, s);
            scan_forward_generic_kernel<T, false><<<(unsigned)gridA, kThreads, 0, s>>>(
                p, n_stations, (const T *)traces, (cx<T> *)spectra, (cx<T> *)scratch);
        }
        ProfScope prof(KID_SCAN_INV, s);
        scan_inverse_generic_kernel<T, false><<<(unsigned)gridB, kThreads, 0, s>>>(
            p, n_stations, n_pairs, (const cx<T> *)spectra, (const cx<T> *)minv, (T *)amp, idx, (cx<T> *)scratch);
    }
    count_launches(2);
    return cudaGetLastError();
}

} // namespace

size_t generic_scratch_bytes(int dtype, int N, long n_units, int upsample)
{
    if (fits_smem(dtype, N, upsample)) return 0;
    return (size_t)generic_grid(n_units) * ((size_t)N + 2 * (size_t)N * upsample) * elem_bytes(dtype);
}

size_t generic_scan_spectra_bytes(int dtype, int K, int n_stations)
{
    return (size_t)n_stations * 2 * K * elem_bytes(dtype);
}

cudaError_t launch_unfold_generic(int dtype, const PlanDev &p, long n_events, int n_stations, const void *traces,
                                  void *efield, void *amp, int32_t *idx, const void *minv, void *scratch, cudaStream_t s,
                                  const UnfoldExt &x)
{
    const long n_units = n_events * (long)n_stations;
    if (n_units <= 0) return cudaSuccess;
    if (x.input_i16)   // int16 ADC counts in, fp32 out
        return launch_unfold_t<float, int16_t>(dtype, p, n_units, n_stations, traces, efield, amp, idx, minv, scratch, s, x);
    return dtype == AERA_F32
               ? launch_unfold_t<float, float>(dtype, p, n_units, n_stations, traces, efield, amp, idx, minv, scratch, s, x)
               : launch_unfold_t<double, double>(dtype, p, n_units, n_stations, traces, efield, amp, idx, minv, scratch, s, x);
}

cudaError_t launch_scan_generic(int dtype, const PlanDev &p, int n_stations, const void *traces, long n_dirs,
                                const void *minv, void *amp, int32_t *idx, void *spectra, void *scratch, cudaStream_t s)
{
    if (n_dirs <= 0 || n_stations <= 0) return cudaSuccess;
    return dtype == AERA_F32
               ? launch_scan_t<float>(dtype, p, n_stations, traces, n_dirs, minv, amp, idx, spectra, scratch, s)
               : launch_scan_t<double>(dtype, p, n_stations, traces, n_dirs, minv, amp, idx, spectra, scratch, s);
}

} // namespace aera

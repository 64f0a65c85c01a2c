// Device-resident reconstruction loop (SURVEY.md 8f "next" row 1; PAPER.md L29 / Fig. 1 and L83):
// the two small steps that close the loop around the unfolding kernels, so that an event batch is
// iterated without leaving the GPU.
//
//   timing_kernel<T>   R19: n_i = lowest n maximising v0[n]^2 + v1[n]^2, w_i = that maximum. One warp per
//                      station, coalesced 16-byte loads, shuffle argmax (lowest index on ties).
//   planefit_kernel<T> R20: weighted plane-wave fit of one event's arrival samples on a flat array,
//                      c n_i / fs = c t0 - (u x_i + v y_i): the weighted means are removed first (two passes
//                      over the event's stations, all in double), which leaves a well-conditioned 2x2
//                      system for (u, v); theta = asin(min(1, |(u,v)|)), phi = atan2(v, u) in [0, 360).
//                      One warp per event; weights are the squared peak amplitudes (or w_i itself for the
//                      voltage timing).
#include "aera_internal.h"

namespace aera {
namespace {

constexpr double kCLight = 299792458.0;

template <typename T> struct Vec4;
template <> struct Vec4<float> { using type = float4; };
template <> struct Vec4<double> { using type = double4; };

template <typename T>
__global__ void __launch_bounds__(256)
timing_kernel(const T *__restrict__ traces, long n_units, int N, int32_t *__restrict__ idx0, T *__restrict__ w0)
{
    const int lane = threadIdx.x & 31;
    const long warp = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const long n_warps = (long)gridDim.x * (blockDim.x >> 5);
    for (long u = warp; u < n_units; u += n_warps) {
        const T *v0 = traces + (size_t)u * 2 * N, *v1 = v0 + N;
        T best = (T)-1; int bi = 0;
        for (int n = 4 * lane; n < N; n += 128) {       // N is a power of two >= 64: whole groups of 4
            T a[4], b[4];
            if constexpr (sizeof(T) == 4) {
                const float4 x = *reinterpret_cast<const float4 *>(v0 + n), y = *reinterpret_cast<const float4 *>(v1 + n);
                a[0] = x.x; a[1] = x.y; a[2] = x.z; a[3] = x.w; b[0] = y.x; b[1] = y.y; b[2] = y.z; b[3] = y.w;
            } else {
                const double2 x0 = *reinterpret_cast<const double2 *>(v0 + n), x1 = *reinterpret_cast<const double2 *>(v0 + n + 2);
                const double2 y0 = *reinterpret_cast<const double2 *>(v1 + n), y1 = *reinterpret_cast<const double2 *>(v1 + n + 2);
                a[0] = x0.x; a[1] = x0.y; a[2] = x1.x; a[3] = x1.y; b[0] = y0.x; b[1] = y0.y; b[2] = y1.x; b[3] = y1.y;
            }
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const T e = a[j] * a[j] + b[j] * b[j];   // (compiled with fmad: one rounding less than the oracle; ties are compared with the index)
                if (e > best) { best = e; bi = n + j; } // ascending n per lane: strict > keeps the lowest index
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const T ob = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
        }
        if (lane == 0) { idx0[u] = bi; w0[u] = best; }
    }
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// square_w: weights are amp^2 (amplitudes given) or w itself (already squared voltages)
template <typename T>
__global__ void __launch_bounds__(128)
planefit_kernel(const double *__restrict__ pos, const int32_t *__restrict__ idx, const T *__restrict__ wsrc, int square_w,
                long n_events, int S, double fs, double *__restrict__ dirs)
{
    const int lane = threadIdx.x & 31;
    const long e = (long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    if (e >= n_events) return;
    const int32_t *ti = idx + (size_t)e * S;
    const T *wi = wsrc + (size_t)e * S;
    const double cs = kCLight / fs;
    double sw = 0, sx = 0, sy = 0, sb = 0;
    for (int i = lane; i < S; i += 32) {
        double w = (double)wi[i]; if (square_w) w *= w;
        if (!(w > 0)) w = 0;
        sw += w; sx += w * pos[2 * i]; sy += w * pos[2 * i + 1]; sb += w * (cs * (double)ti[i]);
    }
    sw = warp_sum(sw); sx = warp_sum(sx); sy = warp_sum(sy); sb = warp_sum(sb);
    double theta = 0.0, phi = 0.0;
    if (sw > 0) {
        const double mx = sx / sw, my = sy / sw, mb = sb / sw;
        double sxx = 0, sxy = 0, syy = 0, sxb = 0, syb = 0;
        for (int i = lane; i < S; i += 32) {
            double w = (double)wi[i]; if (square_w) w *= w;
            if (!(w > 0)) w = 0;
            const double dx = pos[2 * i] - mx, dy = pos[2 * i + 1] - my, db = cs * (double)ti[i] - mb;
            sxx += w * dx * dx; sxy += w * dx * dy; syy += w * dy * dy; sxb += w * dx * db; syb += w * dy * db;
        }
        sxx = warp_sum(sxx); sxy = warp_sum(sxy); syy = warp_sum(syy); sxb = warp_sum(sxb); syb = warp_sum(syb);
        // minimise sum w (db + u dx + v dy)^2 : [sxx sxy; sxy syy] (u, v) = -(sxb, syb)
        const double det = sxx * syy - sxy * sxy;
        if (det != 0.0) {
            const double u = (-sxb * syy + syb * sxy) / det, v = (-syb * sxx + sxb * sxy) / det;
            const double s = hypot(u, v);
            theta = asin(s < 1.0 ? s : 1.0) * (180.0 / 3.14159265358979323846);
            phi = atan2(v, u) * (180.0 / 3.14159265358979323846);
            if (phi < 0) phi += 360.0;
        }
    }
    if (lane == 0) { dirs[2 * e] = theta; dirs[2 * e + 1] = phi; }
}

// first iteration it >= 1 whose direction lies within tol_deg (angle on the sphere) of the previous one, else -1
__global__ void convergence_kernel(const double *__restrict__ dirs_hist, int n_iter, long n_events, double tol_deg, int32_t *__restrict__ conv_iter)
{
    const long e = (long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_events) return;
    const double d2r = 3.14159265358979323846 / 180.0;
    int found = -1;
    double st, ct, sp, cp;
    sincos(dirs_hist[2 * e] * d2r, &st, &ct); sincos(dirs_hist[2 * e + 1] * d2r, &sp, &cp);
    double ax = st * cp, ay = st * sp, az = ct;
    for (int it = 1; it < n_iter; ++it) {
        const double *d = dirs_hist + ((size_t)it * n_events + e) * 2;
        sincos(d[0] * d2r, &st, &ct); sincos(d[1] * d2r, &sp, &cp);
        const double bx = st * cp, by = st * sp, bz = ct;
        const double cx = ay * bz - az * by, cy = az * bx - ax * bz, cz = ax * by - ay * bx;
        const double ang = atan2(sqrt(cx * cx + cy * cy + cz * cz), ax * bx + ay * by + az * bz) / d2r;
        if (found < 0 && ang < tol_deg) found = it;
        ax = bx; ay = by; az = bz;
    }
    conv_iter[e] = found;
}

} // namespace

cudaError_t launch_convergence(const double *dirs_hist, int n_iter, long n_events, double tol_deg, int32_t *conv_iter, cudaStream_t s)
{
    if (n_events <= 0) return cudaSuccess;
    convergence_kernel<<<(unsigned)((n_events + 127) / 128), 128, 0, s>>>(dirs_hist, n_iter, n_events, tol_deg, conv_iter);
    count_launches(1);
    return cudaGetLastError();
}

cudaError_t launch_timing(int dtype, const void *traces, long n_units, int N, int32_t *idx0, void *w0, cudaStream_t s)
{
    if (n_units <= 0) return cudaSuccess;
    ProfScope prof(KID_TIMING, s);
    long grid = (n_units + 7) / 8;
    if (grid > (long)sm_count() * 8) grid = (long)sm_count() * 8;
    if (dtype == AERA_F32) timing_kernel<float><<<(unsigned)grid, 256, 0, s>>>((const float *)traces, n_units, N, idx0, (float *)w0);
    else timing_kernel<double><<<(unsigned)grid, 256, 0, s>>>((const double *)traces, n_units, N, idx0, (double *)w0);
    count_launches(1);
    return cudaGetLastError();
}

cudaError_t launch_planefit(int dtype, const double *pos, const int32_t *idx, const void *w, int square_w, long n_events,
                            int n_stations, double fs, double *dirs, cudaStream_t s)
{
    if (n_events <= 0) return cudaSuccess;
    ProfScope prof(KID_PLANEFIT, s);
    const unsigned grid = (unsigned)((n_events + 3) / 4);
    if (dtype == AERA_F32) planefit_kernel<float><<<grid, 128, 0, s>>>(pos, idx, (const float *)w, square_w, n_events, n_stations, fs, dirs);
    else planefit_kernel<double><<<grid, 128, 0, s>>>(pos, idx, (const double *)w, square_w, n_events, n_stations, fs, dirs);
    count_launches(1);
    return cudaGetLastError();
}

} // namespace aera

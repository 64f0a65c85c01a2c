// Antenna-pattern side of the path (section 3):
//   * repack_kernel : one-time conversion of the user's table into [zenith][azimuth][freq][4]
//   * minv_kernel   : per event (or per scan direction) evaluation of the pattern at the shower
//                     direction for every in-band bin, and inversion of the 2x2 response matrix.
//
// B200 design (differs from the paper's 3-D texture fetch per (f, theta, phi)):
// trilinear interpolation is a tensor product, so the (zenith, azimuth) part is collapsed ONCE per
// direction: the four corner blocks of the repacked table (each a contiguous n_f x 4 complex run,
// 1.3-6.5 KB) are staged into shared memory with four TMA bulk copies (cp.async.bulk + mbarrier),
// blended into one "slab" in double precision, and every in-band bin then needs only a 1-D lerp in
// frequency.  All stations of an event share the direction, so the inverse matrix
// (2/N) H^-1 is built once per event and reused by its stations.  Texture filtering hardware is not
// used: its 8-bit fractional weights explain the paper's +-0.8 % discrepancy (L75) and cannot meet
// the 1e-4 parity bound.
#include "aera_internal.h"
#include "async_copy.cuh"

namespace aera {

template <typename T>
__global__ void repack_kernel(const cx<T> *__restrict__ src, cx<T> *__restrict__ dst, int n_z, int n_a, int n_f)
{
    // src [cp 4][z][a][f]  ->  dst [z][a][f][cp]
    size_t nodes = (size_t)n_z * n_a * n_f;
    size_t total = nodes * 4;
    for (size_t o = blockIdx.x * (size_t)blockDim.x + threadIdx.x; o < total; o += (size_t)gridDim.x * blockDim.x) {
        size_t node = o >> 2;
        int cp = (int)(o & 3);
        dst[o] = src[(size_t)cp * nodes + node];
    }
}

cudaError_t launch_repack(int dtype, const void *src, void *dst, int n_z, int n_a, int n_f, cudaStream_t s)
{
    ProfScope prof(KID_REPACK, s);
    size_t total = (size_t)n_z * n_a * n_f * 4;
    int blocks = (int)((total + 255) / 256);
    if (blocks > sm_count() * 16) blocks = sm_count() * 16;
    if (dtype == AERA_F32)
        repack_kernel<float><<<blocks, 256, 0, s>>>((const cx<float> *)src, (cx<float> *)dst, n_z, n_a, n_f);
    else
        repack_kernel<double><<<blocks, 256, 0, s>>>((const cx<double> *)src, (cx<double> *)dst, n_z, n_a, n_f);
    count_launches(1);
    return cudaGetLastError();
}

struct DirCell {
    int iz, ia0, ia1;
    double w00, w01, w10, w11; // (z, a) corner weights: (iz,ia0) (iz,ia1) (iz+1,ia0) (iz+1,ia1)
};

__device__ inline DirCell direction_cell(const TableGeom &g, double theta, double phi)
{
    DirCell c;
    double zmax = g.z0 + (g.n_z - 1) * g.dz;
    double th = fmin(fmax(theta, g.z0), zmax);
    double uz = (th - g.z0) / g.dz;
    int iz = (int)floor(uz);
    iz = max(0, min(iz, g.n_z - 2));
    double tz = uz - (double)iz;
    int ia0, ia1;
    double ta;
    if (g.periodic) {
        double P = (g.n_a - 1) * g.da;
        double pw = phi - P * floor((phi - g.a0) / P);
        double ua = (pw - g.a0) / g.da;
        double fl = floor(ua);
        ia0 = (int)fl;
        if (ia0 >= g.n_a - 1) ia0 -= (g.n_a - 1);
        if (ia0 < 0) ia0 = 0;
        ta = ua - fl;
        ia1 = (ia0 + 1) % (g.n_a - 1);
    } else {
        double amax = g.a0 + (g.n_a - 1) * g.da;
        double p = fmin(fmax(phi, g.a0), amax);
        double ua = (p - g.a0) / g.da;
        ia0 = (int)floor(ua);
        ia0 = max(0, min(ia0, g.n_a - 2));
        ta = ua - (double)ia0;
        ia1 = ia0 + 1;
    }
    c.iz = iz; c.ia0 = ia0; c.ia1 = ia1;
    c.w00 = (1.0 - tz) * (1.0 - ta);
    c.w01 = (1.0 - tz) * ta;
    c.w10 = tz * (1.0 - ta);
    c.w11 = tz * ta;
    return c;
}

// One CTA per direction. Dynamic smem: [4 corner blocks of n_f*4 cx<T>] [slab n_f*4 cx<double>].
template <typename T>
__global__ void __launch_bounds__(128)
minv_kernel(const cx<T> *__restrict__ table, TableGeom g, const double *__restrict__ dirs,
            const int *__restrict__ bin_if, const double *__restrict__ bin_tf, const double *__restrict__ bin_w, int K, double scale0,
            int layout, int k_lo, int forward, cx<T> *__restrict__ minv, double g0, double g1)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) uint64_t bar;
    __shared__ DirCell cell;

    const int nblk = g.n_f * 4; // complex entries per corner block
    cx<T> *corner = reinterpret_cast<cx<T> *>(smem_raw);
    cx<double> *slab = reinterpret_cast<cx<double> *>(smem_raw + (size_t)4 * nblk * sizeof(cx<T>));
    const long d = blockIdx.x;

    if (threadIdx.x == 0) {
        mbar_init(&bar, 1);
        cell = direction_cell(g, dirs[2 * d], dirs[2 * d + 1]);
        const uint32_t bytes = (uint32_t)(nblk * sizeof(cx<T>));
        mbar_expect_tx(&bar, 4 * bytes);
        const size_t row0 = ((size_t)cell.iz * g.n_a), row1 = ((size_t)(cell.iz + 1) * g.n_a);
        tma_bulk_g2s(corner + 0 * nblk, table + (row0 + cell.ia0) * nblk, bytes, &bar);
        tma_bulk_g2s(corner + 1 * nblk, table + (row0 + cell.ia1) * nblk, bytes, &bar);
        tma_bulk_g2s(corner + 2 * nblk, table + (row1 + cell.ia0) * nblk, bytes, &bar);
        tma_bulk_g2s(corner + 3 * nblk, table + (row1 + cell.ia1) * nblk, bytes, &bar);
    }
    __syncthreads();          // barrier init + cell visible to all
    mbar_wait(&bar, 0);       // the four corner blocks have landed

    // collapse (zenith, azimuth): slab[f][cp] = sum_corners w * H, Re and Im independently, in double
    for (int i = threadIdx.x; i < nblk; i += blockDim.x) {
        double re = cell.w00 * (double)corner[i].re + cell.w01 * (double)corner[nblk + i].re +
                    cell.w10 * (double)corner[2 * nblk + i].re + cell.w11 * (double)corner[3 * nblk + i].re;
        double im = cell.w00 * (double)corner[i].im + cell.w01 * (double)corner[nblk + i].im +
                    cell.w10 * (double)corner[2 * nblk + i].im + cell.w11 * (double)corner[3 * nblk + i].im;
        slab[i].re = re; slab[i].im = im;
    }
    __syncthreads();

    // per in-band bin: 1-D lerp in frequency, invert the 2x2 response, fold in 2/N
    for (int j = threadIdx.x; j < K; j += blockDim.x) {
        const double scale = bin_w ? scale0 * bin_w[j] : scale0;   // pre-filter weight of this bin (aera_pattern_set_band_filter)
        const int jf = bin_if[j];
        const double t = bin_tf[j], t0 = 1.0 - t;
        double hr[4], hi[4];
#pragma unroll
        for (int cp = 0; cp < 4; ++cp) {
            hr[cp] = t0 * slab[jf * 4 + cp].re + t * slab[(jf + 1) * 4 + cp].re;
            hi[cp] = t0 * slab[jf * 4 + cp].im + t * slab[(jf + 1) * 4 + cp].im;
        }
        // h0 = H0theta, h1 = H0phi, h2 = H1theta, h3 = H1phi ; det = h0 h3 - h1 h2
        double dr = (hr[0] * hr[3] - hi[0] * hi[3]) - (hr[1] * hr[2] - hi[1] * hi[2]);
        double di = (hr[0] * hi[3] + hi[0] * hr[3]) - (hr[1] * hi[2] + hi[1] * hr[2]);
        double den = dr * dr + di * di;
        double ir = 0.0, ii = 0.0; // scale / det
        if (den != 0.0) { ir = scale * dr / den; ii = -scale * di / den; }
        cx<T> *o = minv + ((size_t)d * K + j) * 4;
        // E_theta = ( h3 V0 - h1 V1)/det ; E_phi = (-h2 V0 + h0 V1)/det
        cx<T> mt0, mt1, mp0, mp1; // theta <- V0, theta <- V1, phi <- V0, phi <- V1
        // (g0, g1: per-channel input scale, e.g. volts per ADC count of int16 traces: V_c = g_c * raw_c, folded into the columns)
        mt0.re = (T)(g0 * (hr[3] * ir - hi[3] * ii));    mt0.im = (T)(g0 * (hr[3] * ii + hi[3] * ir));
        mt1.re = (T)(-g1 * (hr[1] * ir - hi[1] * ii)); mt1.im = (T)(-g1 * (hr[1] * ii + hi[1] * ir));
        mp0.re = (T)(-g0 * (hr[2] * ir - hi[2] * ii)); mp0.im = (T)(-g0 * (hr[2] * ii + hi[2] * ir));
        mp1.re = (T)(g1 * (hr[0] * ir - hi[0] * ii));    mp1.im = (T)(g1 * (hr[0] * ii + hi[0] * ir));
        if (forward) { // the forward model (aera_fold_batch): scale * H itself, rows (V0 <- E_theta, V0 <- E_phi, V1 <- E_theta, V1 <- E_phi)
            mt0.re = (T)(scale * hr[0]); mt0.im = (T)(scale * hi[0]); mt1.re = (T)(scale * hr[1]); mt1.im = (T)(scale * hi[1]);
            mp0.re = (T)(scale * hr[2]); mp0.im = (T)(scale * hi[2]); mp1.re = (T)(scale * hr[3]); mp1.im = (T)(scale * hi[3]);
        }
        if (layout == MINV_ROWS) {
            o[0] = mt0; o[1] = mt1; o[2] = mp0; o[3] = mp1;
        } else if (layout == MINV_Q4 || layout == MINV_Q2 || layout == MINV_Q1 || layout == MINV_Q8 || layout == MINV_Q16) {
            const int tw = layout == MINV_Q4 ? 4 : (layout == MINV_Q2 ? 2 : (layout == MINV_Q8 ? 8 : (layout == MINV_Q16 ? 16 : 1)));
            const int k = k_lo + j, C = ((k_lo + K - 1) / tw) - (k_lo / tw) + 1;
            cx<T> *q = minv + (size_t)d * 4 * tw * C + (size_t)(k % tw) * 4 * C + ((k / tw) - (k_lo / tw));
            q[0] = mt0; q[C] = mt1; q[2 * C] = mp0; q[3 * C] = mp1;
        } else if (layout == MINV_Q32) {
            const int k = k_lo + j, C = ((k_lo + K - 1) >> 5) - (k_lo >> 5) + 1;
            cx<T> *a = minv + (size_t)d * 128 * C + ((size_t)(k & 31) * 2 * C + ((k >> 5) - (k_lo >> 5))) * 2;
            cx<T> *b = a + (size_t)C * 2;
            a[0].re = mt0.re; a[0].im = mp0.re; a[1].re = mt0.im; a[1].im = mp0.im;
            b[0].re = mt1.re; b[0].im = mp1.re; b[1].re = mt1.im; b[1].im = mp1.im;
        } else if (layout == MINV_PACKED_PAD) {
            const int KP = K + 2 * kMinvPad;
            cx<T> *a = minv + (size_t)d * KP * 4 + (size_t)(j + kMinvPad) * 2, *b = a + (size_t)KP * 2;
            a[0].re = mt0.re; a[0].im = mp0.re; a[1].re = mt0.im; a[1].im = mp0.im;
            b[0].re = mt1.re; b[0].im = mp1.re; b[1].re = mt1.im; b[1].im = mp1.im;
        } else { // MINV_PACKED: two planes per direction, (theta, phi) side by side so a packed
                 // f32x2 load yields both: A[j] = {t0.re, p0.re, t0.im, p0.im}, B[j] = {t1.re, p1.re, t1.im, p1.im}
            cx<T> *a = minv + (size_t)d * K * 4 + (size_t)j * 2, *b = a + (size_t)K * 2;
            a[0].re = mt0.re; a[0].im = mp0.re; a[1].re = mt0.im; a[1].im = mp0.im;
            b[0].re = mt1.re; b[0].im = mp1.re; b[1].re = mt1.im; b[1].im = mp1.im;
        }
    }
    if (layout == MINV_PACKED_PAD) { // the zero pads before and after both planes
        const int KP = K + 2 * kMinvPad;
        const cx<T> z = {(T)0, (T)0};
        for (int j = threadIdx.x; j < kMinvPad; j += blockDim.x) {
            cx<T> *a0 = minv + (size_t)d * KP * 4 + (size_t)j * 2, *a1 = a0 + (size_t)(K + kMinvPad) * 2;
            a0[0] = z; a0[1] = z; a1[0] = z; a1[1] = z;
            a0[(size_t)KP * 2] = z; a0[(size_t)KP * 2 + 1] = z; a1[(size_t)KP * 2] = z; a1[(size_t)KP * 2 + 1] = z;
        }
    }
}

size_t minv_smem_bytes(int dtype, int n_f)
{
    size_t e = dtype == AERA_F32 ? sizeof(cx<float>) : sizeof(cx<double>);
    return (size_t)4 * n_f * 4 * e + (size_t)n_f * 4 * sizeof(cx<double>);
}

cudaError_t launch_minv(int dtype, const void *table, const TableGeom &g, const PlanDev &p,
                        const double *dirs, long n_dirs, void *minv, int layout, double scale, cudaStream_t s, int forward,
                        double g0, double g1)
{
    if (n_dirs <= 0) return cudaSuccess;
    ProfScope prof(KID_MINV, s);
    size_t smem = minv_smem_bytes(dtype, g.n_f);
    cudaError_t e;
    if (dtype == AERA_F32) {
        AERA_ENSURE_DYN_SMEM(minv_kernel<float>, smem);
        minv_kernel<float><<<(unsigned)n_dirs, 128, smem, s>>>((const cx<float> *)table, g, dirs, p.bin_if, p.bin_tf, forward ? nullptr : p.bin_w,
                                                             p.K, scale, layout, p.k_lo, forward, (cx<float> *)minv, g0, g1);
    } else {
        AERA_ENSURE_DYN_SMEM(minv_kernel<double>, smem);
        minv_kernel<double><<<(unsigned)n_dirs, 128, smem, s>>>((const cx<double> *)table, g, dirs, p.bin_if, p.bin_tf, forward ? nullptr : p.bin_w,
                                                              p.K, scale, layout, p.k_lo, forward, (cx<double> *)minv, g0, g1);
    }
    count_launches(1);
    return cudaGetLastError();
}

// aera_unfold_batch_multi: the antenna type of every station, forced into 0 .. n_patterns-1. The unfold kernels index the
// per-table matrix slabs with these values; the caller's array lives on the device and the call is asynchronous, so a bad
// value cannot be reported -- it is made harmless instead (clamped), and the kernels read this copy in the workspace.
__global__ void clamp_pattern_id_kernel(const int32_t *__restrict__ in, int32_t *__restrict__ out, int n, int n_patterns)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = min(max(in[i], 0), n_patterns - 1);
}

cudaError_t launch_clamp_pattern_id(const int32_t *pattern_id, int32_t *out, int n_stations, int n_patterns, cudaStream_t s)
{
    if (n_stations <= 0) return cudaSuccess;
    clamp_pattern_id_kernel<<<(unsigned)((n_stations + 255) / 256), 256, 0, s>>>(pattern_id, out, n_stations, n_patterns);
    count_launches(1);
    return cudaGetLastError();
}

} // namespace aera

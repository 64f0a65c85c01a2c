// Team-per-station fused unfolding kernel for N = 4096, fp64 (BASELINE configs[3]) and fp32 (the same code on plain
// float lanes: a user with 4096-sample fp32 traces gets a register-resident path instead of the generic radix-8 one).
// The team size TW is a template parameter: N = 1024 TW, TW = 4 (described below), 2 (N = 2048: a radix-2 step across
// two warps), 1 (N = 1024: one warp per station, no team exchange), 8 and 16 (N = 8192 / 16384: the radix-TW step across
// the team is a small register FFT, fft_pow2), so fp64 traces of 1024 / 2048 / 8192 samples and fp32 traces of
// 1024 / 8192 / 16384 samples stay register-resident too (fp32 N = 2048 is unfold_w32.cu's). IN16 reads int16 ADC counts.
// Instantiated in unfold_t4k.cu (fp64 + dispatch), unfold_t4k_f32.cu and unfold_t4k_i16.cu.
//
// A "team" of 4 warps (128 threads x 32 complex doubles = 128 registers each) holds one station
// entirely in registers; a CTA runs 2 teams (8 warps, one CTA per SM, persistent). Every long
// transform is 4096 = 4 x 1024: a radix-4 step across the team plus one 1024-point FFT per warp
// (32 x 32 in registers with one shared-memory transpose, fft32.cuh with plain double lanes).
//
//   a1/a2 forward : g[n] = v0[n] + i v1[n] (two real transforms for one). Thread (warp w, lane)
//                   loads g[m + 1024 j'], j' = 0..3, for its 8 values m = lane + 32 (8 w + jj) with
//                   coalesced 8-byte loads, does the 4-point DFT over j' in registers (decimation in
//                   frequency), multiplies y_q[m] by W_4096^{q m}; the team exchanges through shared
//                   memory (lane-preserving, conflict-free) so that warp q owns y_q[0..1023], and
//                   warp q's FFT_1024 gives G[4 k' + q].
//   separation    : 2 V_0[k] = G[k] + conj G[N-k], 2 V_1[k] = -i (G[k] - conj G[N-k]); bin N-k lives
//                   in warp (4-q)&3, so the mirror rows are published through shared memory.
//   a4 solve      : (E_theta, E_phi)[k] = Minv[event][k] (2V_0, 2V_1)[k] on the band rows, in registers;
//                   Minv = (1/N) H^-1 (pattern.cu, once per event) is read through L1/L2 (64 KB per
//                   event at configs[3], shared by the event's 40 stations).
//   a5 inverse    : the mirror image of the forward path. Warp q inverse-transforms its OWN bins
//                   Z[4 k' + q] (zero outside the band rows; E never leaves the registers / tensor memory),
//                   multiplies u_q[m] by W_4096^{-m q}, the team exchanges, and the radix-4 step gives
//                   z[m + 1024 s], s = 0..3, for this thread's 8 values of m: contiguous 8-byte stores.
//                   theta first, then phi (E_phi waits in tensor memory).
//   a6 outputs    : e_p[n] = Re z_p[n] from registers; |z_theta|^2 waits in this lane's tensor-memory
//                   columns (tmem.cuh) for |z_phi|^2; running (max, lowest index) per lane, warp
//                   shuffle argmax, then the 4 warps of the team combine through shared memory.
//   twiddles      : the shared-memory pipe limits this kernel, so geometric twiddle sequences come from
//                   two-term recurrences (reading R18) instead of table reads.
//
// HBM traffic per station: 64 KB read once, 64 KB + 12 B written once.
// The in-band rows (bins k = 4 (lane + 32 row) + q) are template parameters: <4, 12> is configs[3]
// (k = 615..1638).
#pragma once
#include "aera_internal.h"
#include "async_copy.cuh"
#include "fft32.cuh"
#include "tmem.cuh"

namespace aera {
namespace {

// what differs between the two precisions: vector type, lane type for the 32-point FFT, global loads / stores
template <typename T> struct T4k;
template <> struct T4k<double> {
    using T2 = double2; using Lane = LaneF64;
    static __device__ __forceinline__ double ld_stream(const double *p) { double r; asm volatile("ld.global.nc.L1::no_allocate.f64 %0, [%1];" : "=d"(r) : "l"(p)); return r; }
    static __device__ __forceinline__ void st_stream(double *p, double v, unsigned long long pol) { asm volatile("st.global.L2::cache_hint.f64 [%0], %1, %2;" ::"l"(p), "d"(v), "l"(pol) : "memory"); }
    static __device__ __forceinline__ double2 ld_nc2(const double2 *p) { double2 r; asm volatile("ld.global.nc.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p)); return r; }
    static __device__ __forceinline__ unsigned long long bits(double v) { return (unsigned long long)__double_as_longlong(v); }
    static __device__ __forceinline__ double from_bits(unsigned long long b) { return __longlong_as_double((long long)b); }
    static __device__ __forceinline__ double2 make2(double a, double b) { return make_double2(a, b); }
};
template <> struct T4k<float> {
    using T2 = float2; using Lane = LaneF32;
    static __device__ __forceinline__ float ld_stream(const float *p) { float r; asm volatile("ld.global.nc.L1::no_allocate.f32 %0, [%1];" : "=f"(r) : "l"(p)); return r; }
    static __device__ __forceinline__ void st_stream(float *p, float v, unsigned long long pol) { asm volatile("st.global.L2::cache_hint.f32 [%0], %1, %2;" ::"l"(p), "f"(v), "l"(pol) : "memory"); }
    static __device__ __forceinline__ float2 ld_nc2(const float2 *p) { float2 r; asm volatile("ld.global.nc.v2.f32 {%0, %1}, [%2];" : "=f"(r.x), "=f"(r.y) : "l"(p)); return r; }
    static __device__ __forceinline__ unsigned long long bits(float v) { return (unsigned long long)__float_as_uint(v); }
    static __device__ __forceinline__ float from_bits(unsigned long long b) { return __uint_as_float((unsigned)b); }
    static __device__ __forceinline__ float2 make2(float a, float b) { return make_float2(a, b); }
};
// teams per CTA: 2 in fp64 (8 warps x 250 registers; a third team, 168 registers, gains nothing), 4 in fp32 (16 warps x 128)
// (TW < 4: the same number of warps per CTA, i.e. 4 / TW times the teams)
template <typename T> constexpr int kTeamsOf = sizeof(T) == 8 ? 2 : 4;
constexpr int kPlaneBytes = 33 * 32 * 8;              // one warp's padded 32x32 transpose plane (sized for fp64)
// region X of a team = TW planes (33 792 B at TW = 4): exchange buffer / transpose planes / mirror rows
constexpr int kTabF64 = 2 * 1024 * 16;                // T (pass twiddles) + TQ (W_N^t, t < 1024)
constexpr int kCtlF64 = 512;                          // TMEM base, per-team peak slots (teams of 2 or 4 warps: at most 8 teams)

template <typename T>
struct T4kParams {
    using T2 = typename T4k<T>::T2;
    const void *traces;   // T [n_units][2][N], or int16 ADC counts of the same shape (IN16; the counts-to-volts factors are in Minv)
    T *efield;
    T *amp;
    int32_t *idx;
    const T2 *minv;   // [n_events] MINV_Q4 planes [q][entry][C] complex, scaled by 1/N
    const T2 *tw1024; // W_1024^m
    const T2 *twN;    // W_4096^m
    long n_units;
    int n_stations;
    int k_lo, k_hi, K;
    const int32_t *pattern_id;   // [n_stations] antenna type per station, or nullptr (one table)
    size_t minv_pattern_stride;  // double2 elements between the Minv slabs of consecutive tables
};

template <int TW>
__device__ __forceinline__ void team_sync(int team)
{
    if constexpr (TW == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(team + 1), "n"(TW * 32) : "memory");
}
// streamed output with an L2 evict_first policy: the written lines leave the L2 before the L2-prefetched traces do
__device__ __forceinline__ unsigned long long t4k_policy_evict_first()
{
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// W_N^t, N = 1024 TW, for any t in [0, N) from the table of the first 1024 entries: W_4096^{t+1024} = -i W_4096^t,
// W_2048^{t+1024} = -W_2048^t.
template <int TW, typename T2>
__device__ __forceinline__ T2 w4096(const T2 *TQ, int t)
{
    const T2 w = TQ[t & 1023];
    if constexpr (TW == 2) {
        T2 r2 = w;
        if ((t >> 10) & 1) { r2.x = -w.x; r2.y = -w.y; }
        return r2;
    }
    const int quad = (t >> 10) & 3;
    T2 r;
    r.x = (quad & 1) ? w.y : w.x;       // quad 1: -i w = (w.y, -w.x); quad 2: -w; quad 3: i w = (-w.y, w.x)
    r.y = (quad & 1) ? -w.x : w.y;
    if (quad & 2) { r.x = -r.x; r.y = -r.y; }
    return r;
}

// y[k1] *= W_1024^(k1 * lane); "P" plays the real part. The 31 twiddles of a lane are a geometric
// sequence: two interleaved recurrences (even and odd k1, ratio W^{2 lane}) from TWO table reads
// instead of 31. The shared-memory pipe, not the FP64 pipe, limits this kernel; 15 complex
// multiplications per chain cost < 4e-15 of relative accuracy.
template <typename T, typename T2>
__device__ __forceinline__ void pass_twiddle_d(T (&P)[32], T (&Q)[32], const T2 *__restrict__ TW, int lane)
{
    const T2 w1 = TW[32 + lane], w2 = TW[64 + lane];     // W^{lane}, W^{2 lane}
    T er = w2.x, ei = w2.y, orr = w1.x, oi = w1.y;      // current even / odd twiddle
    static_for<1, 32>([&](auto kc) {
        constexpr int k1 = decltype(kc)::value;
        const T wr = (k1 & 1) ? orr : er, wi = (k1 & 1) ? oi : ei;
        T a = P[k1] * wr; a = fma(Q[k1], -wi, a);
        T b = P[k1] * wi; b = fma(Q[k1], wr, b);
        P[k1] = a; Q[k1] = b;
        if constexpr (k1 + 2 < 32) {                         // advance the chain just used by W^{2 lane}
            T nr = wr * w2.x; nr = fma(-wi, w2.y, nr);
            T ni = wr * w2.y; ni = fma(wi, w2.x, ni);
            if (k1 & 1) { orr = nr; oi = ni; } else { er = nr; ei = ni; }
        }
    });
}
template <typename T>
__device__ __forceinline__ void transpose_plane_d(T (&P)[32], T *X, int lane)
{
    static_for<0, 32>([&](auto kc) {
        constexpr int k1 = decltype(kc)::value;
        X[k1 * 33 + lane] = P[k1];
    });
    __syncwarp();
    static_for<0, 32>([&](auto tc) {
        constexpr int t = decltype(tc)::value;
        P[brev5(t)] = X[lane * 33 + t];
    });
    __syncwarp();
}
// 1024-point forward FFT of in[brev5(j)] = x[lane + 32 j]; on return lane k1 holds X[k1 + 32 k2] in
// (P[k2], Q[k2]). Call with (Q, P) for the un-normalised inverse. ONE copy of the 32-point code.
template <typename T, typename T2>
__device__ __forceinline__ void fft1024_d(T (&P)[32], T (&Q)[32], T *X, const T2 *__restrict__ TW, int lane)
{
    int second = 0;
    asm volatile("" : "+r"(second));
#pragma unroll 1
    for (;;) {
        fft32<typename T4k<T>::Lane>(P, Q);
        if (second) break;
        pass_twiddle_d(P, Q, TW, lane);
        transpose_plane_d(P, X, lane);
        transpose_plane_d(Q, X, lane);
        second = 1;
        asm volatile("" : "+r"(second));
    }
}

// R-point forward DFT (R = 2^LOGR <= 32) of the values in (re[i], im[i]), input element j at position brev(j) over LOGR
// bits, output in natural order: the first LOGR stages of fft32's butterfly network (same twiddle indices in units of
// 2 pi / 32). Called with (im, re) it is the un-normalised inverse.
template <class Ln, int LOGR, typename T>
__device__ __forceinline__ void fft_pow2(T *re, T *im)
{
    static_for<0, LOGR>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        constexpr int half = 1 << s;
        static_for<0, (1 << LOGR) / 2>([&](auto bc) {
            constexpr int b = decltype(bc)::value;
            constexpr int j = b & (half - 1);
            constexpr int i0 = ((b - j) << 1) + j;
            constexpr int i1 = i0 + half;
            constexpr int idx = j * (16 >> s);
            butterfly<Ln, idx>(re[i0], im[i0], re[i1], im[i1]);
        });
    });
}
__host__ __device__ constexpr int brev_n(int j, int bits)
{
    int r = 0;
    for (int b = 0; b < bits; ++b) r |= ((j >> b) & 1) << (bits - 1 - b);
    return r;
}

template <typename T, int TW, int RLO, int RHI, bool HAS_EF, int kTeams, bool IN16>
__global__ void __launch_bounds__(kTeams *TW * 32, 1)
unfold_t4k_kernel(T4kParams<T> p)
{
    using T2 = typename T4k<T>::T2;
    using K = T4k<T>;
    static_assert(TW == 1 || TW == 2 || TW == 4 || TW == 8 || TW == 16, "team of 1, 2, 4, 8 or 16 warps");
    static_assert(kTeams * TW <= 16 && (TW == 1 || kTeams <= 15), "tensor-memory column blocks / named barriers");
    constexpr int N = 1024 * TW;
    constexpr int MPW = 32 / TW;                    // values of m per thread in the radix-TW step
    constexpr int kRegionX = TW * kPlaneBytes;
    constexpr int kRows = RHI - RLO + 1;            // band rows per thread (a row = 32 TW bins)
    static_assert(kRows >= 1 && kRows <= 16, "band rows below N/2");
    constexpr int kMirLo = 31 - RHI, kMirHi = (32 - RLO) > 31 ? 31 : (32 - RLO); // rows holding some band bin's mirror
    constexpr int kMirRows = kMirHi - kMirLo + 1;
    static_assert(kMirRows * 512 <= kPlaneBytes, "mirror rows fit region X");
    extern __shared__ __align__(128) unsigned char smem[];
    T2 *TW_ = reinterpret_cast<T2 *>(smem);       // [32][32] pass twiddles W_1024^{k1 t}
    T2 *TQ = TW_ + 1024;                                // W_N^t, t < 1024
    uint32_t *tmem_base = reinterpret_cast<uint32_t *>(smem + kTabF64);
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    constexpr int kLogTW = TW == 16 ? 4 : (TW == 8 ? 3 : (TW == 4 ? 2 : (TW == 2 ? 1 : 0)));
    const int team = warp >> kLogTW, w = warp & (TW - 1);   // (shifts and masks: a signed division hides w's range from the compiler)
    T *peak_v = reinterpret_cast<T *>(smem + kTabF64 + 64) + (TW == 1 ? 0 : team) * (TW < 4 ? 4 : TW);   // [team][TW]
    int *peak_i = reinterpret_cast<int *>(smem + kTabF64 + 64 + (TW == 1 ? 0 : (TW > 4 ? 4 : kTeams)) * 32) + (TW == 1 ? 0 : team) * (TW < 4 ? 4 : TW);   // (unused when TW = 1)
    unsigned char *tb = smem + kTabF64 + kCtlF64 + (size_t)team * kRegionX;
    T *RX = reinterpret_cast<T *>(tb);            // region X
    T *XW = RX + (size_t)w * (kPlaneBytes / 8);        // this warp's transpose plane

    if (warp == 0) tmem_alloc_all(tmem_base);
    for (int i = threadIdx.x; i < 1024; i += blockDim.x) {
        const int k1 = i >> 5, t = i & 31;
        TW_[i] = p.tw1024[(k1 * t) & 1023];
        TQ[i] = p.twN[i];
    }
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tenv = tmem_addr(*tmem_base, warp, (warp >> 2) * 128); // |z_theta|^2: 2 columns per sample, 64 columns
    const uint32_t tephi = tenv + 64;                               // E_phi: 4 columns per band row

    const unsigned long long pol_first = t4k_policy_evict_first();
    const long u0 = p.n_units * (long)blockIdx.x / (long)gridDim.x;
    const long u1 = p.n_units * ((long)blockIdx.x + 1) / (long)gridDim.x;

#pragma unroll 1
    for (long u = u0 + team; u < u1; u += kTeams) {
        const T *v = static_cast<const T *>(p.traces) + (size_t)u * 2 * N;
        const int16_t *v16 = static_cast<const int16_t *>(p.traces) + (size_t)u * 2 * N;
        auto ldv = [&](int i) -> T {   // sample i of the station's [2][N] block
            if constexpr (IN16) { short c; asm volatile("ld.global.nc.L1::no_allocate.s16 %0, [%1];" : "=h"(c) : "l"(v16 + i)); return (T)c; }
            else return K::ld_stream(v + i);
        };
        T *ef = HAS_EF ? p.efield + (size_t)u * 2 * N : nullptr;
        const long ev = u / p.n_stations;
        const T2 *M = p.minv + (size_t)ev * ((size_t)(4 * TW) * ((p.k_hi >> kLogTW) - (p.k_lo >> kLogTW) + 1)) +
                           (p.pattern_id ? (size_t)p.pattern_id[u - ev * p.n_stations] * p.minv_pattern_stride : 0);
        if (w == 0 && lane == 0 && u + kTeams < u1) {
            if (IN16) prefetch_l2_bulk(v16 + (size_t)kTeams * 2 * N, 2 * N * sizeof(int16_t));
            else prefetch_l2_bulk(v + (size_t)kTeams * 2 * N, 2 * N * sizeof(T));
        }

        T P[32], Q[32];
        // ---- a1 + radix-TW step: thread holds y_q[m], q = 0..TW-1, m = lane + 32 (MPW w + jj), at [MPW q + jj]
        if constexpr (TW == 4) {
        static_for<0, 8>([&](auto jc) {
            constexpr int jj = decltype(jc)::value;
            const int m = lane + 32 * (8 * w + jj);
            const T x0r = ldv(m), x1r = ldv(m + 1024);
            const T x2r = ldv(m + 2048), x3r = ldv(m + 3072);
            const T x0i = ldv(N + m), x1i = ldv(N + m + 1024);
            const T x2i = ldv(N + m + 2048), x3i = ldv(N + m + 3072);
            const T ar = x0r + x2r, ai = x0i + x2i, br = x0r - x2r, bi = x0i - x2i;
            const T cr = x1r + x3r, ci = x1i + x3i, dr = x1r - x3r, di = x1i - x3i;
            P[jj] = ar + cr; Q[jj] = ai + ci;                    // y0
            const T y1r = br + di, y1i = bi - dr;           // b - i d
            const T y2r = ar - cr, y2i = ai - ci;
            const T y3r = br - di, y3i = bi + dr;           // b + i d
            const T2 w1 = TQ[m];                            // W_4096^m, m < 1024
            T2 w2, w3;                                      // W^{2m}, W^{3m} by multiplication: one table read, not three
            w2.x = fma(w1.x, w1.x, -(w1.y * w1.y)); w2.y = (w1.x + w1.x) * w1.y;
            w3.x = fma(w2.x, w1.x, -(w2.y * w1.y)); w3.y = fma(w2.x, w1.y, w2.y * w1.x);
            T t;
            t = y1r * w1.x; P[8 + jj] = fma(y1i, -w1.y, t); t = y1r * w1.y; Q[8 + jj] = fma(y1i, w1.x, t);
            t = y2r * w2.x; P[16 + jj] = fma(y2i, -w2.y, t); t = y2r * w2.y; Q[16 + jj] = fma(y2i, w2.x, t);
            t = y3r * w3.x; P[24 + jj] = fma(y3i, -w3.y, t); t = y3r * w3.y; Q[24 + jj] = fma(y3i, w3.x, t);
        });
        } else if constexpr (TW >= 8) {   // radix-TW step as a small register FFT over j'; W_N^{q m} by powers of W_N^m
        static_for<0, MPW>([&](auto jc) {
            constexpr int jj = decltype(jc)::value;
            const int m = lane + 32 * (MPW * w + jj);
            T xr[TW], xi[TW];
            static_for<0, TW>([&](auto tc) {
                constexpr int j = decltype(tc)::value;
                xr[brev_n(j, kLogTW)] = ldv(m + 1024 * j);
                xi[brev_n(j, kLogTW)] = ldv(N + m + 1024 * j);
            });
            fft_pow2<typename K::Lane, kLogTW>(xr, xi);
            const T2 w1 = TQ[m];                            // W_N^m, m < 1024
            T2 wq = w1;
            P[jj] = xr[0]; Q[jj] = xi[0];
            static_for<1, TW>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                T t = xr[q] * wq.x; P[MPW * q + jj] = fma(xi[q], -wq.y, t);
                t = xr[q] * wq.y; Q[MPW * q + jj] = fma(xi[q], wq.x, t);
                if constexpr (q + 1 < TW) {
                    const T nr = fma(wq.x, w1.x, -(wq.y * w1.y)), ni = fma(wq.x, w1.y, wq.y * w1.x);
                    wq.x = nr; wq.y = ni;
                }
            });
        });
        } else if constexpr (TW == 2) {
        static_for<0, 16>([&](auto jc) {
            constexpr int jj = decltype(jc)::value;
            const int m = lane + 32 * (16 * w + jj);
            const T x0r = ldv(m), x1r = ldv(m + 1024);
            const T x0i = ldv(N + m), x1i = ldv(N + m + 1024);
            P[jj] = x0r + x1r; Q[jj] = x0i + x1i;               // y0
            const T y1r = x0r - x1r, y1i = x0i - x1i;
            const T2 w1 = TQ[m];                            // W_2048^m, m < 1024
            T t;
            t = y1r * w1.x; P[16 + jj] = fma(y1i, -w1.y, t); t = y1r * w1.y; Q[16 + jj] = fma(y1i, w1.x, t);
        });
        } else {   // one warp holds the whole station: straight into FFT input order, no exchange
        static_for<0, 32>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            P[brev5(j)] = ldv(lane + 32 * j);
            Q[brev5(j)] = ldv(N + lane + 32 * j);
        });
        }

        // ---- team exchange: warp q collects y_q[lane + 32 j], j = 8 w' + jj, into FFT input order
        team_sync<TW>(team);                                         // region X free (previous station done)
        if constexpr (TW > 1) {
            T *XB = RX;                                     // [q][j][lane]
            static_for<0, 32>([&](auto ic) {
                constexpr int i = decltype(ic)::value;           // i = MPW q + jj
                XB[((i / MPW) * 32 + MPW * w + (i % MPW)) * 32 + lane] = P[i];
            });
            team_sync<TW>(team);
            static_for<0, 32>([&](auto jc) {
                constexpr int j = decltype(jc)::value;
                P[brev5(j)] = XB[(w * 32 + j) * 32 + lane];
            });
            team_sync<TW>(team);
            static_for<0, 32>([&](auto ic) {
                constexpr int i = decltype(ic)::value;
                XB[((i / MPW) * 32 + MPW * w + (i % MPW)) * 32 + lane] = Q[i];
            });
            team_sync<TW>(team);
            static_for<0, 32>([&](auto jc) {
                constexpr int j = decltype(jc)::value;
                Q[brev5(j)] = XB[(w * 32 + j) * 32 + lane];
            });
            team_sync<TW>(team);
        }
        // ---- a2: warp q = w: G[TW (lane + 32 row) + q] in (P[row], Q[row])
        fft1024_d(P, Q, XW, TW_, lane);
        team_sync<TW>(team);                                         // all transposes done: region X becomes the mirror rows
        {
            T2 *PUB = reinterpret_cast<T2 *>(RX);      // [warp][mirror row][lane]
            static_for<kMirLo, kMirHi + 1>([&](auto rc) {
                constexpr int r = decltype(rc)::value;
                PUB[(w * kMirRows + (r - kMirLo)) * 32 + lane] = K::make2(P[r], Q[r]);
            });
        }
        team_sync<TW>(team);
        // ---- separation + a4 on the band rows: E for this warp's bins k = 4 (lane + 32 r) + w, in registers
        T Etr[kRows], Eti[kRows];
        {
            const T2 *PUB = reinterpret_cast<const T2 *>(RX);
            const int C = (p.k_hi >> kLogTW) - (p.k_lo >> kLogTW) + 1;     // Minv columns per (q, entry) plane
            const int pw = (TW - w) & (TW - 1);
            const int plane = (w == 0) ? ((32 - lane) & 31) : (31 - lane);
            const int padd = (w == 0 && lane == 0) ? 1 : 0;      // q = 0, lane 0: mirror row 32 - r
            const T2 *Mq = M + (size_t)w * 4 * C;
            static_for<0, kRows>([&](auto rc) {
                constexpr int i = decltype(rc)::value;
                constexpr int r = RLO + i;
                const int k = TW * (lane + 32 * r) + w;
                const bool inband = k >= p.k_lo && k <= p.k_hi;
                int prow = 31 - r + padd;
                prow = prow > kMirHi ? kMirHi : prow;
                const T2 gm = PUB[(pw * kMirRows + (prow - kMirLo)) * 32 + plane];
                int c = lane + 32 * r - (p.k_lo >> kLogTW);
                c = c < 0 ? 0 : (c > C - 1 ? C - 1 : c);
                const T2 m0 = K::ld_nc2(Mq + c), m1 = K::ld_nc2(Mq + C + c);
                const T2 m2 = K::ld_nc2(Mq + 2 * C + c), m3 = K::ld_nc2(Mq + 3 * C + c);
                const T v0r = P[r] + gm.x, v0i = Q[r] - gm.y;   // 2 V_0
                const T v1r = Q[r] + gm.y, v1i = gm.x - P[r];   // 2 V_1
                T er = m0.x * v0r; er = fma(-m0.y, v0i, er); er = fma(m1.x, v1r, er); er = fma(-m1.y, v1i, er);
                T ei = m0.x * v0i; ei = fma(m0.y, v0r, ei); ei = fma(m1.x, v1i, ei); ei = fma(m1.y, v1r, ei);
                T fr = m2.x * v0r; fr = fma(-m2.y, v0i, fr); fr = fma(m3.x, v1r, fr); fr = fma(-m3.y, v1i, fr);
                T fi = m2.x * v0i; fi = fma(m2.y, v0r, fi); fi = fma(m3.x, v1i, fi); fi = fma(m3.y, v1r, fi);
                Etr[i] = inband ? er : (T)0; Eti[i] = inband ? ei : (T)0;
                // E_phi waits in tensor memory while the registers hold the theta transform
                tmem_st64(tephi + 4 * i, K::bits(inband ? fr : (T)0));
                tmem_st64(tephi + 4 * i + 2, K::bits(inband ? fi : (T)0));
            });
        }
        team_sync<TW>(team);                                         // mirror rows consumed: region X is free for transposes

        // ---- a5/a6: per polarisation, mirror image of the forward path. Warp q inverse-transforms its own
        // bins Z[4 k' + q] (zero outside the band rows), multiplies by W_4096^{-m q}, the team exchanges,
        // and the radix-4 step gives z[m + 1024 s], s = 0..3, for this thread's 8 values of m:
        // contiguous 8-byte stores, 256 bytes per warp instruction.
        T best = (T)-1; int bn = 0;
#pragma unroll 1
        for (int pol = 0; pol < 2; ++pol) {
            if (pol == 0) {
                static_for<0, 32>([&](auto kc) {
                    constexpr int r = decltype(kc)::value;
                    if constexpr (r < RLO || r > RHI) { P[brev5(r)] = (T)0; Q[brev5(r)] = (T)0; }
                    else { P[brev5(r)] = Etr[r - RLO]; Q[brev5(r)] = Eti[r - RLO]; }
                });
            } else {
                unsigned long long ev[2 * kRows];
                static_for<0, kRows>([&](auto rc) {
                    constexpr int i = decltype(rc)::value;
                    ev[2 * i] = tmem_ld64(tephi + 4 * i);
                    ev[2 * i + 1] = tmem_ld64(tephi + 4 * i + 2);
                });
                tmem_wait_ld();
                static_for<0, kRows>([&](auto rc) {
                    constexpr int i = decltype(rc)::value;
                    tmem_ld_dep(ev[2 * i], ev[2 * i + 1]);
                });
                static_for<0, 32>([&](auto kc) {
                    constexpr int r = decltype(kc)::value;
                    if constexpr (r < RLO || r > RHI) { P[brev5(r)] = (T)0; Q[brev5(r)] = (T)0; }
                    else {
                        P[brev5(r)] = K::from_bits(ev[2 * (r - RLO)]);
                        Q[brev5(r)] = K::from_bits(ev[2 * (r - RLO) + 1]);
                    }
                });
            }
            fft1024_d(Q, P, XW, TW_, lane);                        // inverse: roles swapped; u_q[m = lane + 32 b] in (P[b], Q[b])
            if (w != 0) {
                // u_q[m] conj(W_4096^{q m}), m = lane + 32 b: two interleaved recurrences over b (ratio W^{64 q})
                T2 r2, c0, c1;
                if constexpr (TW >= 8) {   // three values per transform: straight from the plan's full table W_N^t
                    r2 = p.twN[(64 * w) & (N - 1)]; c0 = p.twN[(w * lane) & (N - 1)]; c1 = p.twN[(w * (lane + 32)) & (N - 1)];
                } else {
                    r2 = w4096<TW>(TQ, 64 * w);
                    c0 = w4096<TW>(TQ, (w * lane) & (N - 1)); c1 = w4096<TW>(TQ, (w * (lane + 32)) & (N - 1));
                }
                T er = c0.x, ei = c0.y, orr = c1.x, oi = c1.y;
                static_for<0, 32>([&](auto bc) {
                    constexpr int b = decltype(bc)::value;
                    const T wr = (b & 1) ? orr : er, wi = (b & 1) ? oi : ei;
                    const T ur = P[b], ui = Q[b];
                    T a = ur * wr; a = fma(ui, wi, a);
                    T c = ui * wr; c = fma(ur, -wi, c);
                    P[b] = a; Q[b] = c;
                    if constexpr (b + 2 < 32) {
                        T nr = wr * r2.x; nr = fma(-wi, r2.y, nr);
                        T ni = wr * r2.y; ni = fma(wi, r2.x, ni);
                        if (b & 1) { orr = nr; oi = ni; } else { er = nr; ei = ni; }
                    }
                });
            }
            team_sync<TW>(team);                                     // all transposes done: region X is the exchange buffer
            if constexpr (TW > 1) {
                T *XB = RX;                                 // [q][b][lane]
                static_for<0, 32>([&](auto bc) {
                    constexpr int b = decltype(bc)::value;
                    XB[(w * 32 + b) * 32 + lane] = P[b];
                });
                team_sync<TW>(team);
                static_for<0, 32>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;       // i = MPW q + jj
                    P[i] = XB[((i / MPW) * 32 + MPW * w + (i % MPW)) * 32 + lane];
                });
                team_sync<TW>(team);
                static_for<0, 32>([&](auto bc) {
                    constexpr int b = decltype(bc)::value;
                    XB[(w * 32 + b) * 32 + lane] = Q[b];
                });
                team_sync<TW>(team);
                static_for<0, 32>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    Q[i] = XB[((i / MPW) * 32 + MPW * w + (i % MPW)) * 32 + lane];
                });
                team_sync<TW>(team);
            }
            // radix-TW step (inverse sign): z_s = sum_q (+i)^{s q} u_q (TW = 4), left in place at [MPW s + jj]
            if constexpr (TW == 2) {
                static_for<0, 16>([&](auto jc) {
                    constexpr int jj = decltype(jc)::value;
                    const T ar = P[jj], ai = Q[jj];
                    P[jj] = ar + P[16 + jj]; Q[jj] = ai + Q[16 + jj];
                    P[16 + jj] = ar - P[16 + jj]; Q[16 + jj] = ai - Q[16 + jj];
                });
            }
            if constexpr (TW >= 8) {
                static_for<0, MPW>([&](auto jc) {
                    constexpr int jj = decltype(jc)::value;
                    T xr[TW], xi[TW];
                    static_for<0, TW>([&](auto qc) {
                        constexpr int q = decltype(qc)::value;
                        xr[brev_n(q, kLogTW)] = P[MPW * q + jj]; xi[brev_n(q, kLogTW)] = Q[MPW * q + jj];
                    });
                    fft_pow2<typename K::Lane, kLogTW>(xi, xr);          // inverse: roles swapped
                    static_for<0, TW>([&](auto sc2) {
                        constexpr int sidx = decltype(sc2)::value;
                        P[MPW * sidx + jj] = xr[sidx]; Q[MPW * sidx + jj] = xi[sidx];
                    });
                });
            }
            if constexpr (TW == 4)
            static_for<0, 8>([&](auto jc) {
                constexpr int jj = decltype(jc)::value;
                const T ar = P[jj] + P[16 + jj], ai = Q[jj] + Q[16 + jj];
                const T br = P[jj] - P[16 + jj], bi = Q[jj] - Q[16 + jj];
                const T cr = P[8 + jj] + P[24 + jj], ci = Q[8 + jj] + Q[24 + jj];
                const T dr = P[8 + jj] - P[24 + jj], di = Q[8 + jj] - Q[24 + jj];
                P[jj] = ar + cr; Q[jj] = ai + ci;
                P[8 + jj] = br - di; Q[8 + jj] = bi + dr;        // b + i d
                P[16 + jj] = ar - cr; Q[16 + jj] = ai - ci;
                P[24 + jj] = br + di; Q[24 + jj] = bi - dr;      // b - i d
            });
            // outputs: index i = MPW s + jj is sample n = lane + 32 (MPW w + jj) + 1024 s (ascending in i)
            const int nbase = lane + 32 * MPW * w;
            if (pol == 0) {
                static_for<0, 32>([&](auto ic) {
                    constexpr int i = decltype(ic)::value;
                    if (HAS_EF) K::st_stream(ef + nbase + 32 * (i % MPW) + 1024 * (i / MPW), P[i], pol_first);
                    T e2 = P[i] * P[i]; e2 = fma(Q[i], Q[i], e2);
                    tmem_st64(tenv + 2 * i, K::bits(e2));
                });
                tmem_wait_st();
            } else {
                static_for<0, 4>([&](auto cc) {
                    constexpr int c = decltype(cc)::value;
                    unsigned long long ev[8];
                    static_for<0, 8>([&](auto jc) {
                        constexpr int j = decltype(jc)::value;
                        ev[j] = tmem_ld64(tenv + 2 * (8 * c + j));
                    });
                    tmem_wait_ld();
                    static_for<0, 4>([&](auto jc) {
                        constexpr int j = decltype(jc)::value;
                        tmem_ld_dep(ev[2 * j], ev[2 * j + 1]);
                    });
                    static_for<0, 8>([&](auto jc) {
                        constexpr int j = decltype(jc)::value;
                        constexpr int i = 8 * c + j;
                        const int n = nbase + 32 * (i % MPW) + 1024 * (i / MPW);
                        if (HAS_EF) K::st_stream(ef + N + n, P[i], pol_first);
                        T e2 = fma(P[i], P[i], K::from_bits(ev[j]));
                        e2 = fma(Q[i], Q[i], e2);
                        if (e2 > best) { best = e2; bn = n; }
                    });
                });
            }
        }
        // ---- a6: lane -> warp -> team argmax, lowest index on ties in every stage
        int bi = bn;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const T ob = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
        }
        if constexpr (TW == 1) {
            if (lane == 0) { p.amp[u] = sqrt(best); p.idx[u] = bi; }
            continue;
        }
        if (lane == 0) { peak_v[w] = best; peak_i[w] = bi; }
        team_sync<TW>(team);
        if (w == 0 && lane == 0) {
            T bv = peak_v[0]; int bx = peak_i[0];
#pragma unroll
            for (int i = 1; i < TW; ++i)
                if (peak_v[i] > bv || (peak_v[i] == bv && peak_i[i] < bx)) { bv = peak_v[i]; bx = peak_i[i]; }
            p.amp[u] = sqrt(bv); p.idx[u] = bx;
        }
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_free_all(*tmem_base);
}

template <typename T, int TW, int RLO, int RHI, bool HAS_EF, bool IN16 = false>
cudaError_t launch_t4k(const T4kParams<T> &q, cudaStream_t s)
{
    constexpr int kTeams = kTeamsOf<T> * 4 / TW;       // the same warps per CTA for every team size
    const size_t smem = (size_t)kTabF64 + kCtlF64 + (size_t)kTeams * TW * kPlaneBytes;
    auto kern = unfold_t4k_kernel<T, TW, RLO, RHI, HAS_EF, kTeams, IN16>;
    AERA_ENSURE_DYN_SMEM(kern, smem);
    long grid = (q.n_units + kTeams - 1) / kTeams;
    if (grid > sm_count()) grid = sm_count();
    kern<<<(unsigned)grid, kTeams * TW * 32, smem, s>>>(q);
    return cudaGetLastError();
}

// IN16: the instantiations that read int16 ADC counts (fp32 only; their own translation unit)
template <typename T, bool IN16 = false>
cudaError_t launch_t4k_typed(const PlanDev &p, long n_units, int n_stations, const void *traces, void *efield, void *amp, int32_t *idx,
                             const void *minv, cudaStream_t s, const UnfoldExt &x)
{
    using T2 = typename T4k<T>::T2;
    T4kParams<T> q;
    q.traces = traces; q.efield = (T *)efield; q.amp = (T *)amp; q.idx = idx;
    q.minv = (const T2 *)minv; q.tw1024 = (const T2 *)p.tw1024; q.twN = (const T2 *)p.twN;
    q.n_units = n_units; q.n_stations = n_stations; q.k_lo = p.k_lo; q.k_hi = p.k_hi; q.K = p.K;
    q.pattern_id = x.pattern_id; q.minv_pattern_stride = x.minv_pattern_stride;
    // rows 4..12 of 32 TW bins (30-80 MHz at fs = 200 MHz for every N; configs[3]) have their own instantiation; <0, 15> serves
    // any other band
    const int tw = p.N / 1024;
    const bool r412 = (p.k_lo / (32 * tw)) == 4 && (p.k_hi / (32 * tw)) == 12;
    auto pick = [&](auto twc) -> cudaError_t {
        constexpr int TWc = decltype(twc)::value;
        if (r412) return efield ? launch_t4k<T, TWc, 4, 12, true, IN16>(q, s) : launch_t4k<T, TWc, 4, 12, false, IN16>(q, s);
        return efield ? launch_t4k<T, TWc, 0, 15, true, IN16>(q, s) : launch_t4k<T, TWc, 0, 15, false, IN16>(q, s);
    };
    if (tw == 1) return pick(IC<1>{});
    if (tw == 8) return pick(IC<8>{});
    if constexpr (sizeof(T) == 4) {     // (sixteen fp64 warps of 250 registers do not fit an SM)
        if (tw == 16) return pick(IC<16>{});
    }
    if constexpr (sizeof(T) == 8) {     // (fp32 N = 2048 is the warp kernel's)
        if (tw == 2) return pick(IC<2>{});
    }
    return pick(IC<4>{});
}

} // namespace

} // namespace aera

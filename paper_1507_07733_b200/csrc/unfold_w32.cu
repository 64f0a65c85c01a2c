// Warp-per-station fused unfolding kernel for N = 2048 fp32 (BASELINE configs[1], the headline).
//
// One warp owns one station at a time and never synchronises with another warp. Every transform is a
// 1024-point complex FFT done as 32 x 32: each lane runs a 32-point FFT in registers (fft32.cuh),
// the warp transposes through shared memory once, each lane runs a second 32-point FFT. Two
// transforms ride in the two halves of the packed f32x2 lanes:
//
//   a1/a2 forward : g_r[m] = v0[2m+r] + i v1[2m+r], r = 0,1 in the two lanes. An 8-byte load of
//                   channel 0 IS the packed real part, of channel 1 the packed imaginary part.
//                   G_r = FFT_1024(g_r).  With the mirror bin 1024-k (one exchange through shared
//                   memory) the four real polyphase spectra separate, and
//                   2 V_c[k] = F'_c0[k] + W_2048^k F'_c1[k]   (k < 1024 covers the whole band).
//   a4 solve      : (E_theta, E_phi)[k] = Minv[event][k] (V_0, V_1)[k]; Minv = (1/N) H^-1 comes from
//                   pattern.cu once per event, laid out as (theta, phi) pairs so E lands packed.
//   a5 inverse    : the analytic spectrum is zero above N/2, so z[2m+s] = IFFT_1024(E[k] W_2048^{-sk}),
//                   s = 0,1: two packed (theta, phi) transforms instead of two 2048-point ones.
//                   The inverse is the forward routine with the re/im arrays swapped.
//   a6 outputs    : e_p[n] = Re z_p[n] straight from registers; env^2 = |z_theta|^2 + |z_phi|^2 and a
//                   running (max, lowest index) per lane, then a 5-step shuffle reduction.
//
// HBM traffic per station: 16 KB read once (L2-prefetched one station ahead with
// cp.async.bulk.prefetch.L2), 16 KB + 8 B written once. Shared memory per warp: one 8.25 KB padded
// transpose buffer + a stash for the in-band spectrum (needed twice, s = 0 and 1).
#include "aera_internal.h"
#include "fft32.cuh"

namespace aera {
namespace {

using L = LaneF32x2;
using R = F2;

constexpr int kM = 1024;
constexpr int kXElems = 33 * 32; // padded 32x32 transpose buffer, 8-byte elements

struct W32Params {
    const float *traces;
    float *efield;
    float *amp;
    int32_t *idx;
    const float4 *minv;   // [n_events][K][2] float4: {t0re,p0re,t0im,p0im} {t1re,p1re,t1im,p1im}
    const float2 *tw1024; // W_1024^m
    const float2 *twN;    // W_2048^m
    long n_units;
    int n_stations;
    int k_lo, k_hi, K;
    int stash_slots;      // per-warp stash capacity in 512-byte slots (>= max(band rows, mirror rows))
};

__device__ __forceinline__ R ld_stream_b64(const void *p)
{
    R r;
    asm volatile("ld.global.nc.L1::no_allocate.b64 %0, [%1];" : "=l"(r.v) : "l"(p));
    return r;
}
__device__ __forceinline__ float4 ld_nc_f4(const float4 *p)
{
    float4 r;
    asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ void prefetch_l2_bulk(const void *p, unsigned bytes)
{
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}

// y[k1] *= W_1024^(k1 * lane) ; T[k1*32 + lane] holds the twiddle (re, im). "A" plays the real part.
__device__ __forceinline__ void pass_twiddle(R (&A)[32], R (&B)[32], const float2 *__restrict__ T, int lane)
{
    static_for<1, 32>([&](auto kc) {
        constexpr int k1 = decltype(kc)::value;
        const float2 w = T[k1 * 32 + lane];
        const R wr = L::bc(w.x), wi = L::bc(w.y), nwi = L::bc(-w.y);
        R a = L::mul(A[k1], wr);
        a = L::fma(B[k1], nwi, a);
        R b = L::mul(A[k1], wi);
        b = L::fma(B[k1], wr, b);
        A[k1] = a; B[k1] = b;
    });
}

// 32x32 transpose of one register plane through the padded buffer: value k1 of lane t goes to lane
// k1, which receives it as input element t of its second-pass FFT (stored at position brev5(t)).
__device__ __forceinline__ void transpose_plane(R (&P)[32], R *X, int lane)
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

// Full 1024-point forward FFT of the packed data held as in[brev5(j)] = x[lane + 32 j].
// On return lane k1 holds X[k1 + 32 k2] in (A[k2], B[k2]). Call with (B, A) for the inverse.
__device__ __forceinline__ void fft1024(R (&A)[32], R (&B)[32], R *X, const float2 *__restrict__ T, int lane)
{
    fft32<L>(A, B);
    pass_twiddle(A, B, T, lane);
    transpose_plane(A, X, lane);
    transpose_plane(B, X, lane);
    fft32<L>(A, B);
}

__device__ __forceinline__ void peak_update(float e2, int n, float &best, int &bi)
{
    if (e2 > best || (e2 == best && n < bi)) { best = e2; bi = n; }
}

// Outputs of one inverse transform: lane a, register b holds z[m = a + 32 b] of (theta, phi);
// sample index n = 2 m + parity.
__device__ __forceinline__ void emit(const R (&zr)[32], const R (&zi)[32], int lane, int parity, float *ef,
                                     float &best, int &bi)
{
    static_for<0, 32>([&](auto bc) {
        constexpr int b = decltype(bc)::value;
        const int n = 2 * (lane + 32 * b) + parity;
        float rt, rp;
        L::unpack(zr[b], rt, rp);
        if (ef) { ef[n] = rt; ef[2 * kM + n] = rp; }
        R q = L::mul(zr[b], zr[b]);
        q = L::fma(zi[b], zi[b], q);
        float qt, qp;
        L::unpack(q, qt, qp);
        peak_update(qt + qp, n, best, bi);
    });
}

template <int WARPS>
__global__ void __launch_bounds__(WARPS * 32, 1)
unfold_w32_kernel(W32Params p)
{
    extern __shared__ __align__(16) unsigned char smem[];
    float2 *T = reinterpret_cast<float2 *>(smem);               // [32][32] pass twiddles
    float2 *TS = T + 1024;                                       // [1024] W_2048^k
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const size_t per_warp = (size_t)kXElems * 8 + (size_t)p.stash_slots * 512;
    unsigned char *wbase = smem + 2 * 1024 * sizeof(float2) + (size_t)warp * per_warp;
    R *X = reinterpret_cast<R *>(wbase);                         // transpose buffer
    float4 *Q = reinterpret_cast<float4 *>(wbase);               // mirror exchange (overlays X + stash)
    float4 *ST = reinterpret_cast<float4 *>(wbase + (size_t)kXElems * 8); // stash [slot][lane] (re, im) packed

    for (int i = threadIdx.x; i < 1024; i += blockDim.x) {
        const int k1 = i >> 5, t = i & 31;
        T[i] = p.tw1024[(k1 * t) & 1023];
        TS[i] = p.twN[i];
    }
    __syncthreads();

    const int k2lo = p.k_lo >> 5, k2hi = p.k_hi >> 5;                 // rows of in-band bins
    const int mlo = (kM - p.k_hi) >> 5, mhi = (kM - p.k_lo) >> 5;     // rows of their mirror bins
    const long gw = (long)blockIdx.x * WARPS + warp, nw = (long)gridDim.x * WARPS;

    for (long u = gw; u < p.n_units; u += nw) {
        const float *v = p.traces + (size_t)u * 4 * kM;
        float *ef = p.efield ? p.efield + (size_t)u * 4 * kM : nullptr;
        const float4 *Mv = p.minv + ((size_t)(u / p.n_stations) * p.K) * 2;
        if (lane == 0 && u + nw < p.n_units) prefetch_l2_bulk(v + (size_t)nw * 4 * kM, 4 * kM * sizeof(float));

        // ---- a1: the station's two traces, read once, straight into FFT input order
        R A[32], B[32];
        static_for<0, 32>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            A[brev5(j)] = ld_stream_b64(v + 2 * (lane + 32 * j));            // (v0[2m], v0[2m+1])
            B[brev5(j)] = ld_stream_b64(v + 2 * kM + 2 * (lane + 32 * j));   // (v1[2m], v1[2m+1])
        });

        // ---- a2: forward FFT of g_0, g_1
        fft1024(A, B, X, T, lane);

        // ---- mirror exchange: publish the rows that are somebody's bin 1024-k
        static_for<0, 32>([&](auto rc) {
            constexpr int r = decltype(rc)::value;
            if (r >= mlo && r <= mhi) {
                float ax, ay, bx, by;
                L::unpack(A[r], ax, ay); L::unpack(B[r], bx, by);
                Q[(r - mlo) * 32 + lane] = make_float4(ax, ay, bx, by);
            }
        });
        __syncwarp();

        // ---- separate channels, fold the two polyphase halves, a4: E = Minv V
        R Zr[32], Zi[32]; // inverse-transform input, element k2 at brev5(k2)
        static_for<0, 32>([&](auto kc) {
            constexpr int k2 = decltype(kc)::value;
            R er = L::zero(), ei = L::zero();
            if (k2 >= k2lo && k2 <= k2hi) {
                const int k = lane + 32 * k2;
                if (k >= p.k_lo && k <= p.k_hi) {
                    // partner bin 1024-k lives in lane (32-lane)&31, row 31-k2 (row 32-k2 for lane 0)
                    const int prow = (lane == 0 ? 32 - k2 : 31 - k2) - mlo;
                    const float4 pq = Q[prow * 32 + ((32 - lane) & 31)];
                    const R pr = L::pack(pq.x, pq.y), pi = L::pack(pq.z, pq.w);
                    // F'_0 = G + conj(Gm) = 2 FFT(v0 polyphase r), F'_1 = -i (G - conj(Gm)) = 2 FFT(v1 polyphase r)
                    const R f0r = L::add(A[k2], pr), f0i = L::sub(B[k2], pi);
                    const R f1r = L::add(B[k2], pi), f1i = L::sub(pr, A[k2]);
                    float f0r0, f0r1, f0i0, f0i1, f1r0, f1r1, f1i0, f1i1;
                    L::unpack(f0r, f0r0, f0r1); L::unpack(f0i, f0i0, f0i1);
                    L::unpack(f1r, f1r0, f1r1); L::unpack(f1i, f1i0, f1i1);
                    const float2 w = TS[k]; // W_2048^k = (wr, wi)
                    // 2 V_c = F'_c(r=0) + W F'_c(r=1)
                    float v0r = fmaf(w.x, f0r1, f0r0); v0r = fmaf(-w.y, f0i1, v0r);
                    float v0i = fmaf(w.x, f0i1, f0i0); v0i = fmaf(w.y, f0r1, v0i);
                    float v1r = fmaf(w.x, f1r1, f1r0); v1r = fmaf(-w.y, f1i1, v1r);
                    float v1i = fmaf(w.x, f1i1, f1i0); v1i = fmaf(w.y, f1r1, v1i);
                    const float4 m0 = ld_nc_f4(Mv + 2 * (k - p.k_lo)), m1 = ld_nc_f4(Mv + 2 * (k - p.k_lo) + 1);
                    const R Ma = L::pack(m0.x, m0.y), Mb = L::pack(m0.z, m0.w), Mc = L::pack(m1.x, m1.y), Md = L::pack(m1.z, m1.w);
                    er = L::mul(Ma, L::bc(v0r)); er = L::fma(Mb, L::bc(-v0i), er);
                    er = L::fma(Mc, L::bc(v1r), er); er = L::fma(Md, L::bc(-v1i), er);
                    ei = L::mul(Ma, L::bc(v0i)); ei = L::fma(Mb, L::bc(v0r), ei);
                    ei = L::fma(Mc, L::bc(v1i), ei); ei = L::fma(Md, L::bc(v1r), ei);
                }
            }
            Zr[brev5(k2)] = er; Zi[brev5(k2)] = ei;
        });
        __syncwarp(); // all mirror reads done before the stash overwrites the region

        // ---- stash E for the odd-sample transform
        static_for<0, 32>([&](auto kc) {
            constexpr int k2 = decltype(kc)::value;
            if (k2 >= k2lo && k2 <= k2hi) {
                float a, b, c, d;
                L::unpack(Zr[brev5(k2)], a, b); L::unpack(Zi[brev5(k2)], c, d);
                ST[(k2 - k2lo) * 32 + lane] = make_float4(a, b, c, d);
            }
        });

        float best = -1.0f; int bi = 0x7fffffff;

        // ---- a5/a6: even samples  z[2m] = IFFT_1024(E)
        fft1024(Zi, Zr, X, T, lane);
        emit(Zr, Zi, lane, 0, ef, best, bi);

        // ---- odd samples  z[2m+1] = IFFT_1024(E W_2048^-k)
        static_for<0, 32>([&](auto kc) {
            constexpr int k2 = decltype(kc)::value;
            R er = L::zero(), ei = L::zero();
            if (k2 >= k2lo && k2 <= k2hi) {
                const float4 s = ST[(k2 - k2lo) * 32 + lane];
                const float2 w = TS[lane + 32 * k2];
                const R sr = L::pack(s.x, s.y), si = L::pack(s.z, s.w);
                // (sr + i si)(wr - i wi)
                er = L::mul(sr, L::bc(w.x)); er = L::fma(si, L::bc(w.y), er);
                ei = L::mul(si, L::bc(w.x)); ei = L::fma(sr, L::bc(-w.y), ei);
            }
            Zr[brev5(k2)] = er; Zi[brev5(k2)] = ei;
        });
        fft1024(Zi, Zr, X, T, lane);
        emit(Zr, Zi, lane, 1, ef, best, bi);

        // ---- a6: warp argmax, lowest index on ties
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float ob = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ob > best || (ob == best && oi < bi)) { best = ob; bi = oi; }
        }
        if (lane == 0) { p.amp[u] = sqrtf(best); p.idx[u] = bi; }
        __syncwarp();
    }
}

constexpr int kWarps = 8;

} // namespace

bool w32_supported(int dtype, const PlanDev &p)
{
    return dtype == AERA_F32 && p.N == 2 * kM && p.k_hi < kM && p.k_lo >= 1;
}

static int w32_slots(const PlanDev &p)
{
    const int band_rows = (p.k_hi >> 5) - (p.k_lo >> 5) + 1;
    const int mirror_rows = ((kM - p.k_lo) >> 5) - ((kM - p.k_hi) >> 5) + 1;
    // the mirror exchange overlays transpose buffer + stash: needs mirror_rows*512 <= 8448 + slots*512
    int need = mirror_rows - (kXElems * 8) / 512;
    return band_rows > need ? band_rows : need;
}

cudaError_t launch_unfold_w32(const PlanDev &p, long n_events, int n_stations, const void *traces, void *efield,
                              void *amp, int32_t *idx, const void *minv, cudaStream_t s)
{
    const long n_units = n_events * (long)n_stations;
    if (n_units <= 0) return cudaSuccess;
    ProfScope prof(KID_UNFOLD, s);
    W32Params q;
    q.traces = (const float *)traces; q.efield = (float *)efield; q.amp = (float *)amp; q.idx = idx;
    q.minv = (const float4 *)minv; q.tw1024 = (const float2 *)p.tw1024; q.twN = (const float2 *)p.twN;
    q.n_units = n_units; q.n_stations = n_stations; q.k_lo = p.k_lo; q.k_hi = p.k_hi; q.K = p.K;
    q.stash_slots = w32_slots(p);
    const size_t smem = 2 * 1024 * sizeof(float2) + (size_t)kWarps * ((size_t)kXElems * 8 + (size_t)q.stash_slots * 512);
    cudaError_t e = cudaFuncSetAttribute(unfold_w32_kernel<kWarps>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    long grid = (n_units + kWarps - 1) / kWarps;
    if (grid > 148) grid = 148;
    unfold_w32_kernel<kWarps><<<(unsigned)grid, kWarps * 32, smem, s>>>(q);
    count_launches(1);
    return cudaGetLastError();
}

} // namespace aera

// Long-trace fused unfolding kernel for N = 65536 fp32 (BASELINE configs[4]):
// a multi-pass transform whose intermediates live in an L2-resident per-station scratch. One station per
// thread-block CLUSTER of 8 CTAs x 4 warps (32 warps: every phase below is one round of 32 warp tasks),
// three CTAs of three different stations per SM (12 warps whose phases are decoupled), persistent;
// every warp-level piece is shared with the N = 2048 kernel (w32_common.cuh: 32-point register FFTs,
// 1024-point warp FFTs, packed f32x2 lanes).
//
// One station's complex buffer (512 KB) is beyond an SM's shared memory (227 KB) and distributed
// shared memory is slower than L2 on this part (~21 B/clk/SM against ~43 B/clk/SM of L2), so the
// passes exchange through global memory that stays in the 126 MB L2: <= 55 clusters x 0.96 MB.
//
//   phase 1 (32 warp tasks)  a1 + first forward pass. g_r[m] = v0[2m+r] + i v1[2m+r], r = 0,1 in the two
//       packed halves (an 8-byte load of channel 0 IS the packed real part), m = mm + 1024 j'. Task mb:
//       lane mm = lane + 32 mb loads j' = 0..31, 32-point FFT over j' in registers, times W_32768^{q mm},
//       stores y_q[mm] to scratch Y[q][mm].
//   phase 2 (16 pair tasks)  second forward pass + separation + a4. Warp q: FFT_1024 over mm gives
//       G_r[32 k' + q]; the mirror bin 32768 - k lives in warp 32 - q, so warps (q, 32-q) form a pair and
//       swap their mirror rows through shared memory; 2 V_c[k] = F'_c0[k] + W_N^k F'_c1[k];
//       E = Minv V on the band rows (Minv: pattern.cu, once per event, plane layout MINV_Q32);
//       E (theta, phi packed) goes to scratch E[q][k'].
//   a5: K <= N/4, so z[4 m' + s] = IFFT_16384 over k < 16384 of E[k] W_N^{-s k}, s = 0..3 (quarter-pruned),
//       done for s in pairs (2h, 2h+1) so the 512 KB of Y can be reused for the pair's intermediates:
//   phase 3 (32 warp tasks per pair)  task (s, q'): IFFT_1024 over k'' of E[16 k'' + q'] W_N^{-s k},
//       times W_16384^{-mm q'}, to scratch U[s&1][q'][mm].
//   phase 4 (32 warp tasks per pair)  a6. Task mb: lane mm loads U[.][q'][mm], q' = 0..15, for both s of
//       the pair, 16-point inverse FFT over q' gives z[4 (mm + 1024 t) + s], t = 0..15: e_p = Re z_p as
//       8-byte (s = 2h, 2h+1) pairs, env^2 = |z_theta|^2 + |z_phi|^2 running argmax, then a 64-bit
//       shared-memory atomicMax of (env^2 bits, ~index) across the CTA's tasks.
//
// HBM traffic per station: 512 KB read once, 512 KB + 8 B written once (the first pair's Re z is parked
// in the scratch so that the second pass stores whole 16-byte quads). L2 traffic per station: ~5 MB (the real roofline of this kernel, with the FP32 pipe).
#include <cstdio>
#include <cstdlib>
#include "w32_common.cuh"

namespace aera {
namespace {

constexpr int kLN = 65536;
constexpr int kLWarps = 4;                 // warps per CTA
constexpr int kLCtasPerSm = 3;             // 12 warps per SM, from three different stations (phases decoupled)
constexpr int kLCluster = 8;               // CTAs per station (thread-block cluster): 32 warps, every phase (32 tasks) is ONE round
inline int long_max_clusters() { return sm_count() * kLCtasPerSm / kLCluster; }   // 55 stations in flight on 148 SMs
constexpr int kLTeam = kLWarps * kLCluster;
constexpr size_t kYBytes = (size_t)32 * 1024 * 16;            // Y[q][mm] two 8-byte planes; reused as U[2][16][1024]
// band geometry of an instantiation: phase 2 rows P2LO..P2HI (k' >> 5, k' = k >> 5, i.e. k >> 10) and phase 3 rows
// 2 P2LO .. 2 P2HI + 1 (k'' >> 5, k'' = k >> 4, i.e. k >> 9). <1, 12> is configs[4] (k = 1311 .. 13107); <0, 15> serves
// any other band below N/4.
template <int P2LO, int P2HI>
struct LongGeom {
    static constexpr int kP2Lo = P2LO, kP2Hi = P2HI;
    static constexpr int kP3Lo = 2 * P2LO, kP3Hi = 2 * P2HI + 1;
    static constexpr int kMirLoL = 31 - P2HI, kMirRowsL = 32 - kMirLoL;   // mirror rows published to the pair partner
    static_assert(P2LO >= 0 && P2HI <= 15 && 2 * kMirRowsL * 256 <= kXBytes, "rows below N/4; mirror rows fit the warp buffer");
};

struct LongParams {
    const float *traces;
    float *efield;
    float *amp;
    int32_t *idx;
    const float4 *minv;    // [n_events] MINV_Q32: [q 32][plane A|B][C] float4
    const float2 *tw1024;  // W_1024^m
    const float2 *twN;     // W_65536^m
    unsigned char *scratch; // [gridDim.x] { Y 512 KB | E 32 x C x 16 B }
    size_t scratch_stride;
    long n_units;
    int n_stations;
    int k_lo, k_hi, K, C;  // C = (k_hi >> 5) - (k_lo >> 5) + 1
    const int32_t *pattern_id;   // [n_stations] antenna type per station, or nullptr (one table)
    size_t minv_pattern_stride;  // float4 elements between the Minv slabs of consecutive tables
};

// L2 residency: the scratch (<= 55 x 0.96 MB) must stay in the 126 MB L2 while 1 MB per station streams
// through it, so scratch accesses carry an evict_last policy and the streamed traces / E-field an
// evict_first policy (createpolicy + .L2::cache_hint).
__device__ __forceinline__ unsigned long long policy_evict_last()
{
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ unsigned long long policy_evict_first()
{
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// scratch: L2-only loads (written by other warps of this CTA), evict_last
__device__ __forceinline__ R ld_sc(const void *p, unsigned long long pol)
{
    R r;
    asm volatile("ld.global.cg.L2::cache_hint.b64 %0, [%1], %2;" : "=l"(r.v) : "l"(p), "l"(pol) : "memory");
    return r;
}
__device__ __forceinline__ void st_sc(void *p, R v, unsigned long long pol)
{
    asm volatile("st.global.cg.L2::cache_hint.b64 [%0], %1, %2;" ::"l"(p), "l"(v.v), "l"(pol) : "memory");
}
__device__ __forceinline__ R ld_stream_pol(const void *p, unsigned long long pol)
{
    R r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::cache_hint.b64 %0, [%1], %2;" : "=l"(r.v) : "l"(p), "l"(pol));
    return r;
}
__device__ __forceinline__ void st_stream_f4(void *p, float4 v, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;"
                 ::"l"(p), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}

// W_65536^x from two 256-entry tables: W^x = TA[x >> 8] TB[x & 255] (one complex multiplication in fp32).
__device__ __forceinline__ float2 w64k(const float2 *TA, const float2 *TB, unsigned x)
{
    const float2 a = TA[(x >> 8) & 255], b = TB[x & 255];
    float2 r;
    r.x = fmaf(a.x, b.x, -(a.y * b.y));
    r.y = fmaf(a.x, b.y, a.y * b.x);
    return r;
}
// (re, im) *= (wr + i wi), packed lanes, scalar twiddle
__device__ __forceinline__ void cmul_packed(R &re, R &im, float wr, float wi)
{
    R a = L::mul(re, L::bc(wr)); a = L::fma(im, L::bc(-wi), a);
    R b = L::mul(re, L::bc(wi)); b = L::fma(im, L::bc(wr), b);
    re = a; im = b;
}
// one copy of the 32-point code for both passes of a 1024-point transform (see unfold_w32.cu)
__device__ __forceinline__ void fft1024_loop(R (&A)[32], R (&B)[32], R *X, const float2 *__restrict__ T, int lane)
{
    int second = 0;
    asm volatile("" : "+r"(second));
#pragma unroll 1
    for (;;) {
        fft32<L>(A, B);
        if (second) break;
        pass_twiddle(A, B, T, lane);
        transpose_plane(A, X, lane);
        transpose_plane(B, X, lane);
        second = 1;
        asm volatile("" : "+r"(second));
    }
}
// all threads of the cluster; orders global-memory accesses between its CTAs (release / acquire)
__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\nbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ unsigned cluster_rank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ float2 cmulf(float2 a, float2 b)
{
    float2 r;
    r.x = fmaf(a.x, b.x, -(a.y * b.y));
    r.y = fmaf(a.x, b.y, a.y * b.x);
    return r;
}
__device__ __forceinline__ void pair_sync(int pair)
{
    asm volatile("bar.sync %0, 64;" ::"r"(pair + 1) : "memory");
}

// 16-point inverse FFT (sign +) on packed lanes, natural order in and out: two radix-4 stages.
__device__ __forceinline__ void ifft4(R &x0r, R &x0i, R &x1r, R &x1i, R &x2r, R &x2i, R &x3r, R &x3i)
{
    const R ar = L::add(x0r, x2r), ai = L::add(x0i, x2i), br = L::sub(x0r, x2r), bi = L::sub(x0i, x2i);
    const R cr = L::add(x1r, x3r), ci = L::add(x1i, x3i), dr = L::sub(x1r, x3r), di = L::sub(x1i, x3i);
    x0r = L::add(ar, cr); x0i = L::add(ai, ci);
    x1r = L::sub(br, di); x1i = L::add(bi, dr);      // b + i d
    x2r = L::sub(ar, cr); x2i = L::sub(ai, ci);
    x3r = L::add(br, di); x3i = L::sub(bi, dr);      // b - i d
}
__device__ __forceinline__ void ifft16(R (&xr)[16], R (&xi)[16])
{
    // x[q], q = 4 a + b: stage 1 over a (stride 4) for each b, twiddle W_16^{-b c}, stage 2 over b
    static_for<0, 4>([&](auto bc) {
        constexpr int b = decltype(bc)::value;
        ifft4(xr[b], xi[b], xr[4 + b], xi[4 + b], xr[8 + b], xi[8 + b], xr[12 + b], xi[12 + b]); // -> c = 0..3 at [4 c + b]
    });
    static_for<1, 4>([&](auto cc) {
        constexpr int c = decltype(cc)::value;
        static_for<1, 4>([&](auto bc) {
            constexpr int b = decltype(bc)::value;
            constexpr int e = (b * c) & 15;                     // times exp(+2 pi i e / 16)
            constexpr float wr = (float)kCos32[(2 * e) & 15] * ((2 * e) & 16 ? -1.f : 1.f);
            constexpr float wi = (float)kSin32[(2 * e) & 15] * ((2 * e) & 16 ? -1.f : 1.f);
            cmul_packed(xr[4 * c + b], xi[4 * c + b], wr, wi);
        });
    });
    static_for<0, 4>([&](auto cc) {
        constexpr int c = decltype(cc)::value;
        ifft4(xr[4 * c], xi[4 * c], xr[4 * c + 1], xi[4 * c + 1], xr[4 * c + 2], xi[4 * c + 2], xr[4 * c + 3], xi[4 * c + 3]); // -> t = c + 4 d at [4 c + d]
    });
}

template <bool HAS_EF, int P2LO, int P2HI>
__global__ void __cluster_dims__(kLCluster, 1, 1) __launch_bounds__(kLWarps * 32, kLCtasPerSm)
unfold_long_f32_kernel(LongParams p)
{
    using LG = LongGeom<P2LO, P2HI>;
    constexpr int kP2Lo = LG::kP2Lo, kP2Hi = LG::kP2Hi, kP3Lo = LG::kP3Lo, kP3Hi = LG::kP3Hi;
    constexpr int kMirLoL = LG::kMirLoL, kMirRowsL = LG::kMirRowsL;
    extern __shared__ __align__(128) unsigned char smem[];
    float2 *T = reinterpret_cast<float2 *>(smem);                       // [32][32] pass twiddles W_1024^{k1 t}
    float2 *TA = T + 1024;                                              // W_N^{256 a}
    float2 *TB = TA + 256;                                              // W_N^{b}
    unsigned long long *peak = reinterpret_cast<unsigned long long *>(TB + 256);
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const int crank = (int)cluster_rank();
    const int gw = crank * kLWarps + warp;                              // warp index within the station's team of 32
    const long cluster_id = blockIdx.x / kLCluster, n_clusters = gridDim.x / kLCluster;
    R *X = reinterpret_cast<R *>(smem + 8192 + 4096 + 128 + (size_t)warp * kXBytes);   // transpose plane / mirror rows
    R *Xpartner = reinterpret_cast<R *>(smem + 8192 + 4096 + 128 + (size_t)(warp ^ 1) * kXBytes);

    for (int i = threadIdx.x; i < 1024; i += blockDim.x) {
        const int k1 = i >> 5, t = i & 31;
        T[i] = p.tw1024[(k1 * t) & 1023];
    }
    for (int i = threadIdx.x; i < 256; i += blockDim.x) {
        TA[i] = p.twN[256 * i];
        TB[i] = p.twN[i];
    }
    if (threadIdx.x == 0) *peak = 0ull;
    __syncthreads();

    unsigned char *sc = p.scratch + (size_t)cluster_id * p.scratch_stride;
    unsigned long long *gpeak = reinterpret_cast<unsigned long long *>(sc + p.scratch_stride - 64);  // [2] per-CTA peaks
    R *YA = reinterpret_cast<R *>(sc), *YB = YA + 32 * 1024;
    R *EA = reinterpret_cast<R *>(sc + kYBytes), *EB = EA + 32 * p.C;
    R *H0 = EB + 32 * p.C;                                              // [pol 2][t 16][mm 1024] parked (s = 0, 1) pairs
    R *U0 = H0 + 2 * 16 * 1024;                                         // U[2][16][1024] two 8-byte planes
    const int C = p.C, c_lo = p.k_lo >> 5;
    const unsigned long long pol_last = policy_evict_last(), pol_first = policy_evict_first();

    // ---------------- phase 1 of station uu: loads + 32-point transform over j' + twiddle -> Y. It depends on nothing but
    // the free Y buffer, so it runs in the same round as phase 4 of the previous station (no barrier between them).
    auto phase1 = [&](long uu) {
        const float *v0 = p.traces + (size_t)uu * 2 * kLN, *v1 = v0 + kLN;
#pragma unroll 1
        for (int mb = gw; mb < 32; mb += kLTeam) {
            const int mm = lane + 32 * mb;
            R A[32], B[32];
            static_for<0, 32>([&](auto jc) {
                constexpr int j = decltype(jc)::value;
                A[brev5(j)] = ld_stream_pol(v0 + 2 * (mm + 1024 * j), pol_first);
                B[brev5(j)] = ld_stream_pol(v1 + 2 * (mm + 1024 * j), pol_first);
            });
            fft32<L>(A, B);
            // W_32768^{q mm} = W_N^{2 q mm}: geometric in q; recurrences of 8 steps re-seeded from the table
            const float2 rat = w64k(TA, TB, (unsigned)(2 * mm));
            float2 w = rat;
            static_for<0, 32>([&](auto qc) {
                constexpr int q = decltype(qc)::value;
                if constexpr (q > 0) {
                    if constexpr ((q & 7) == 0) w = w64k(TA, TB, (unsigned)(2 * q * mm));
                    cmul_packed(A[q], B[q], w.x, w.y);
                    if constexpr ((q & 7) != 7) w = cmulf(w, rat);
                }
                st_sc(YA + q * 1024 + mm, A[q], pol_last);
                st_sc(YB + q * 1024 + mm, B[q], pol_last);
            });
        }
    };
    if (cluster_id < p.n_units) phase1(cluster_id);
    cluster_sync_all();

#pragma unroll 1
    for (long u = cluster_id; u < p.n_units; u += n_clusters) {
        float *ef = HAS_EF ? p.efield + (size_t)u * 2 * kLN : nullptr;
        const long ev = u / p.n_stations;
        const float4 *Mev = p.minv + (size_t)ev * 64 * C + (p.pattern_id ? (size_t)p.pattern_id[u - ev * p.n_stations] * p.minv_pattern_stride : 0);

        // ---------------- phase 2: 1024-point transform per q, separation with the pair partner, fold, a4 -> E
#pragma unroll 1
        for (int pt = gw >> 1; pt < 16; pt += kLTeam / 2) {
            const int role = warp & 1;
            const int q = pt == 0 ? 16 * role : (role ? 32 - pt : pt);
            R A[32], B[32];
            static_for<0, 32>([&](auto jc) {
                constexpr int j = decltype(jc)::value;
                A[brev5(j)] = ld_sc(YA + q * 1024 + lane + 32 * j, pol_last);
                B[brev5(j)] = ld_sc(YB + q * 1024 + lane + 32 * j, pol_last);
            });
            fft1024_loop(A, B, X, T, lane);     // lane k1, register k2: G_r[32 (k1 + 32 k2) + q], r = 0,1 packed
            static_for<kMirLoL, 32>([&](auto rc) {
                constexpr int r = decltype(rc)::value;
                X[(r - kMirLoL) * 32 + lane] = A[r];
                X[(kMirRowsL + r - kMirLoL) * 32 + lane] = B[r];
            });
            pair_sync(warp >> 1);
            const R *PUB = pt == 0 ? X : Xpartner;      // q = 0 and q = 16 are their own mirrors
            const int plane = q == 0 ? ((32 - lane) & 31) : (31 - lane);
            const int padd = (q == 0 && lane == 0) ? 1 : 0;
            const float4 *MA = Mev + (size_t)(2 * q) * C, *MB = MA + C;
            const float2 rat = TA[4];                                // W_N^{1024}: k grows by 1024 per row
            float2 w = make_float2(1.f, 0.f);
            static_for<kP2Lo, kP2Hi + 1>([&](auto rc) {
                constexpr int k2 = decltype(rc)::value;
                if constexpr (((k2 - kP2Lo) % 6) == 0) w = w64k(TA, TB, (unsigned)(32 * (lane + 32 * k2) + q));   // W_N^k
                else w = cmulf(w, rat);
                const int kp = lane + 32 * k2, k = 32 * kp + q;
                const bool inband = k >= p.k_lo && k <= p.k_hi;
                int prow = 31 - k2 + padd - kMirLoL;
                if (kP2Lo == 0 && prow > kMirRowsL - 1) prow = kMirRowsL - 1;   // (k = 0, whose mirror row would be 32, is never in band)
                const R ar = A[k2], ai = B[k2], pr = PUB[prow * 32 + plane], pi = PUB[(kMirRowsL + prow) * 32 + plane];
                const R f0r = L::add(ar, pr), f0i = L::sub(ai, pi);
                const R f1r = L::add(ai, pi), f1i = L::sub(pr, ar);
                float f0r0, f0r1, f0i0, f0i1, f1r0, f1r1, f1i0, f1i1;
                L::unpack(f0r, f0r0, f0r1); L::unpack(f0i, f0i0, f0i1);
                L::unpack(f1r, f1r0, f1r1); L::unpack(f1i, f1i0, f1i1);
                float v0r = fmaf(w.x, f0r1, f0r0); v0r = fmaf(-w.y, f0i1, v0r);
                float v0i = fmaf(w.x, f0i1, f0i0); v0i = fmaf(w.y, f0r1, v0i);
                float v1r = fmaf(w.x, f1r1, f1r0); v1r = fmaf(-w.y, f1i1, v1r);
                float v1i = fmaf(w.x, f1i1, f1i0); v1i = fmaf(w.y, f1r1, v1i);
                const int c = kp - c_lo;
                const int cc = c < 0 ? 0 : (c > C - 1 ? C - 1 : c);
                const float4 m0 = ld_nc_f4(MA + cc), m1 = ld_nc_f4(MB + cc);
                const R Ma = L::pack(m0.x, m0.y), Mb = L::pack(m0.z, m0.w), Mc = L::pack(m1.x, m1.y), Md = L::pack(m1.z, m1.w);
                R er = L::mul(Ma, L::bc(v0r)); er = L::fma(Mb, L::bc(-v0i), er);
                er = L::fma(Mc, L::bc(v1r), er); er = L::fma(Md, L::bc(-v1i), er);
                R ei = L::mul(Ma, L::bc(v0i)); ei = L::fma(Mb, L::bc(v0r), ei);
                ei = L::fma(Mc, L::bc(v1i), ei); ei = L::fma(Md, L::bc(v1r), ei);
                if (!inband) { er = L::zero(); ei = L::zero(); }
                if (c >= 0 && c < C) { st_sc(EA + q * C + c, er, pol_last); st_sc(EB + q * C + c, ei, pol_last); }
            });
            pair_sync(warp >> 1);                       // mirror rows consumed before the next transposes
        }
        cluster_sync_all();

        R *UA = U0, *UB = U0 + 32 * 1024;               // U[sl][q'][mm] (index (16 sl + q') * 1024 + mm), its own buffer:
                                                        // Y is being refilled by the next station's phase 1 meanwhile
        float best = -1.0f; int bn = 0;
#pragma unroll 1
        for (int h = 0; h < 2; ++h) {
            // ---------------- phase 3: task (s = 2h + sl, q'): pruned inverse 1024-point transform -> U
#pragma unroll 1
            for (int ti = gw; ti < 32; ti += kLTeam) {
                const int sl = ti >> 4, qp = ti & 15, s = 2 * h + sl;
                const int q = qp + 16 * (lane & 1);                 // bin k = 16 k'' + q' = 32 k' + q
                R A[32], B[32];                                      // inverse roles: A = Im, B = Re
                const float2 rin = w64k(TA, TB, (unsigned)(512 * s));     // k grows by 512 per row
                float2 win = make_float2(1.f, 0.f);
                static_for<0, 32>([&](auto jc) {
                    constexpr int j = decltype(jc)::value;
                    if constexpr (j < kP3Lo || j > kP3Hi) { A[brev5(j)] = L::zero(); B[brev5(j)] = L::zero(); }
                    else {
                        const int kpp = lane + 32 * j;
                        const int c = (kpp >> 1) - c_lo;
                        R er = L::zero(), ei = L::zero();
                        if (c >= 0 && c < C) { er = ld_sc(EA + q * C + c, pol_last); ei = ld_sc(EB + q * C + c, pol_last); }
                        if (s != 0) {                                // E[k] conj(W_N^{s k}), recurrences of 8 rows
                            if constexpr (((j - kP3Lo) & 7) == 0) win = w64k(TA, TB, (unsigned)(s * (16 * kpp + qp)));
                            else win = cmulf(win, rin);
                            cmul_packed(er, ei, win.x, -win.y);
                        }
                        B[brev5(j)] = er; A[brev5(j)] = ei;
                    }
                });
                fft1024_loop(A, B, X, T, lane);                      // lane a, register b: u[mm = a + 32 b] = B + i A
                const float2 rout = w64k(TA, TB, (unsigned)(128 * qp)); // mm grows by 32 per register
                float2 wout = make_float2(1.f, 0.f);
                static_for<0, 32>([&](auto bc) {
                    constexpr int b = decltype(bc)::value;
                    const int mm = lane + 32 * b;
                    if (qp != 0) {                                   // conj(W_16384^{mm q'}) = conj(W_N^{4 mm q'})
                        if constexpr ((b & 7) == 0) wout = w64k(TA, TB, (unsigned)(4 * qp * mm));
                        else wout = cmulf(wout, rout);
                        cmul_packed(B[b], A[b], wout.x, -wout.y);
                    }
                    st_sc(UA + (16 * sl + qp) * 1024 + mm, B[b], pol_last);
                    st_sc(UB + (16 * sl + qp) * 1024 + mm, A[b], pol_last);
                });
            }
            cluster_sync_all();
            // ---------------- phase 4: task mb: 16-point inverse transforms over q' for s = 2h, 2h+1; outputs
#pragma unroll 1
            for (int mb = gw; mb < 32; mb += kLTeam) {
                const int mm = lane + 32 * mb;
                R re0[16];
                static_for<0, 2>([&](auto sc_) {
                    constexpr int sl = decltype(sc_)::value;
                    R xr[16], xi[16];
                    static_for<0, 16>([&](auto qc) {
                        constexpr int qp = decltype(qc)::value;
                        xr[qp] = ld_sc(UA + (16 * sl + qp) * 1024 + mm, pol_last);
                        xi[qp] = ld_sc(UB + (16 * sl + qp) * 1024 + mm, pol_last);
                    });
                    ifft16(xr, xi);                                  // [4 c + d] holds t = c + 4 d
                    static_for<0, 16>([&](auto ic) {
                        constexpr int i = decltype(ic)::value;
                        constexpr int t = (i >> 2) + 4 * (i & 3);
                        const int n = 4 * (mm + 1024 * t) + 2 * h + sl;
                        R qq = L::mul(xr[i], xr[i]); qq = L::fma(xi[i], xi[i], qq);
                        float qt, qf; L::unpack(qq, qt, qf);
                        const float e2 = qt + qf;
                        if (e2 > best || (e2 == best && n < bn)) { best = e2; bn = n; }
                        if (sl == 0) re0[i] = xr[i];
                        else if (HAS_EF) {
                            // Re z of the four sample phases of one 16-byte quad come from two passes (h = 0, 1):
                            // pass 0 parks its (s = 0, 1) pairs in the L2-resident scratch, pass 1 stores whole
                            // quads, so every 32-byte sector of the E-field is written once and in full.
                            float t0, p0, t1, p1;
                            L::unpack(re0[i], t0, p0); L::unpack(xr[i], t1, p1);
                            R *hp = H0 + (size_t)t * 1024 + mm;
                            if (h == 0) {
                                st_sc(hp, L::pack(t0, t1), pol_last);
                                st_sc(hp + 16 * 1024, L::pack(p0, p1), pol_last);
                            } else {
                                const R a = ld_sc(hp, pol_last), b = ld_sc(hp + 16 * 1024, pol_last);
                                float a0, a1, b0, b1;
                                L::unpack(a, a0, a1); L::unpack(b, b0, b1);
                                st_stream_f4(ef + (n - 3), make_float4(a0, a1, t0, t1), pol_first);
                                st_stream_f4(ef + kLN + (n - 3), make_float4(b0, b1, p0, p1), pol_first);
                            }
                        }
                    });
                });
            }
            if (h == 0) cluster_sync_all();                          // U is rewritten by the next pair's phase 3
        }
        // ---------------- phase 1 of the next station, in the same round as this station's last phase 4
        if (u + n_clusters < p.n_units) phase1(u + n_clusters);
        // ---------------- a6: lane -> warp -> CTA argmax (lowest index on ties: key = value bits, ~index)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const float ob = __shfl_xor_sync(0xffffffffu, best, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bn, o);
            if (ob > best || (ob == best && oi < bn)) { best = ob; bn = oi; }
        }
        if (lane == 0)
            atomicMax(peak, ((unsigned long long)__float_as_uint(best) << 32) | (unsigned long long)(0xffffffffu - (unsigned)bn));
        __syncthreads();
        if (threadIdx.x == 0) {                                      // this CTA's peak -> the cluster's slot
            asm volatile("st.global.cg.u64 [%0], %1;" ::"l"(gpeak + crank), "l"(*peak) : "memory");
            *peak = 0ull;
        }
        cluster_sync_all();                                          // also: Y of the next station is complete, U is free
        if (crank == 0 && threadIdx.x == 0) {
            unsigned long long key = 0ull;
#pragma unroll
            for (int c = 0; c < kLCluster; ++c) {
                unsigned long long kc;
                asm volatile("ld.global.cg.u64 %0, [%1];" : "=l"(kc) : "l"(gpeak + c) : "memory");
                key = kc > key ? kc : key;
            }
            p.amp[u] = sqrtf(__uint_as_float((unsigned)(key >> 32)));
            p.idx[u] = (int)(0xffffffffu - (unsigned)(key & 0xffffffffu));
        }
    }
}

} // namespace

bool long_f32_supported(int dtype, const PlanDev &p)
{
    // any band below N/4 (the inverse transforms are quarter-pruned); configs[4]'s rows (20-200 MHz at fs = 1 GHz) have
    // their own instantiation
    return dtype == AERA_F32 && p.N == kLN && p.k_lo >= 1 && p.k_hi < kLN / 4;
}

static size_t long_stride(const PlanDev &p)
{
    const size_t C = (size_t)((p.k_hi >> 5) - (p.k_lo >> 5) + 1);
    return (2 * kYBytes + 2 * 32 * C * 8 + 2 * 16 * 1024 * 8 + 64 + 255) & ~(size_t)255;   // Y | E | parked pairs | U | per-CTA peaks
}
// megabytes of persisting-L2 carve-out requested through aera_set_long_trace_l2_persist; -1 = leave the device's limit alone
static std::atomic<long> g_long_persist_mb{-1};
long set_long_persist_mb(long mb) { return g_long_persist_mb.exchange(mb < 0 ? -1 : mb); }

size_t long_f32_scratch_bytes(const PlanDev &p) { return long_max_clusters() * long_stride(p); }

cudaError_t launch_unfold_long_f32(const PlanDev &p, long n_events, int n_stations, const void *traces, void *efield,
                                   void *amp, int32_t *idx, const void *minv, void *scratch, cudaStream_t s, const UnfoldExt &x)
{
    const long n_units = n_events * (long)n_stations;
    if (n_units <= 0) return cudaSuccess;
    ProfScope prof(KID_UNFOLD, s);
    LongParams q;
    q.traces = (const float *)traces; q.efield = (float *)efield; q.amp = (float *)amp; q.idx = idx;
    q.minv = (const float4 *)minv; q.tw1024 = (const float2 *)p.tw1024; q.twN = (const float2 *)p.twN;
    q.scratch = (unsigned char *)scratch; q.scratch_stride = long_stride(p);
    q.n_units = n_units; q.n_stations = n_stations; q.k_lo = p.k_lo; q.k_hi = p.k_hi; q.K = p.K;
    q.C = (p.k_hi >> 5) - (p.k_lo >> 5) + 1;
    q.pattern_id = x.pattern_id; q.minv_pattern_stride = x.minv_pattern_stride / 2;   // complex float -> float4 elements
    const size_t smem = 8192 + 4096 + 128 + (size_t)kLWarps * kXBytes;
    cudaError_t e;
    auto launch = [&](auto kern) -> cudaError_t {
        AERA_ENSURE_DYN_SMEM(kern, smem);
        // persistent clusters: as many as can be co-resident (a cluster of 8 must fit one GPC), at most one per station
        static std::atomic<int> max_clusters_of[kMaxDevices];   // cached per device (same for both instantiations to within rounding)
        const int slot = device_slot();
        int max_clusters = slot >= 0 ? max_clusters_of[slot].load(std::memory_order_relaxed) : 0;
        if (max_clusters == 0) {
            cudaLaunchConfig_t cfg = {};
            cfg.gridDim = dim3(kLCluster * long_max_clusters()); cfg.blockDim = dim3(kLWarps * 32); cfg.dynamicSmemBytes = smem;
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = kLCluster; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            cfg.attrs = at; cfg.numAttrs = 1;
            int n = 0;
            if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess || n <= 0) { (void)cudaGetLastError(); n = long_max_clusters(); }
            max_clusters = n < long_max_clusters() ? n : long_max_clusters();
            if (slot >= 0) max_clusters_of[slot].store(max_clusters, std::memory_order_relaxed);
        }
        const long clusters = n_units < max_clusters ? n_units : max_clusters;
        // The scratch lines carry an evict_last policy, which holds only inside the persisting carve-out of the L2: without
        // one a fifth of the scratch writes are evicted to DRAM before being overwritten (measured 1.83 MB of DRAM traffic
        // per station against 1.05 MB algorithmic, 1.146 M stations/s; with a 79 MB carve-out 1.11 MB, 1.116 M stations/s;
        // with 70 MB = the scratch size 1.23 MB, 1.135 M stations/s). The carve-out is device-wide state that belongs to
        // the caller, so it is only touched on request: aera_set_long_trace_l2_persist (include/aera_unfold.h).
        const long want_mb = g_long_persist_mb.load(std::memory_order_relaxed);
        if (want_mb >= 0) {
            static std::atomic<long> applied_mb[kMaxDevices];   // request last applied on each device, + 1 (0 = none yet)
            if (slot < 0 || applied_mb[slot].load(std::memory_order_relaxed) != want_mb + 1) {
                int mx = 0, dev = 0;
                (void)cudaGetDevice(&dev);
                (void)cudaDeviceGetAttribute(&mx, cudaDevAttrMaxPersistingL2CacheSize, dev);
                size_t want = (size_t)want_mb << 20;
                if (want > (size_t)mx) want = (size_t)mx;
                if (cudaDeviceSetLimit(cudaLimitPersistingL2CacheSize, want) != cudaSuccess) (void)cudaGetLastError();
                if (slot >= 0) applied_mb[slot].store(want_mb + 1, std::memory_order_relaxed);
            }
        }
        kern<<<(unsigned)(kLCluster * clusters), kLWarps * 32, smem, s>>>(q);
        return cudaGetLastError();
    };
    if ((p.k_lo >> 10) == 1 && (p.k_hi >> 10) == 12)
        e = efield ? launch(unfold_long_f32_kernel<true, 1, 12>) : launch(unfold_long_f32_kernel<false, 1, 12>);
    else
        e = efield ? launch(unfold_long_f32_kernel<true, 0, 15>) : launch(unfold_long_f32_kernel<false, 0, 15>);
    count_launches(1);
    return e;
}

} // namespace aera

// Building blocks shared by the warp-per-station kernels (unfold_w32.cu, scan_w32.cu): N = 2048 fp32,
// every transform a 1024-point complex FFT done as 32 x 32 (fft32.cuh) with two transforms riding in
// the two halves of the packed f32x2 lanes. See unfold_w32.cu for the derivation of each step.
#pragma once
#include "aera_internal.h"
#include "async_copy.cuh"
#include "fft32.cuh"
#include "tmem.cuh"

namespace aera {
namespace {

using L = LaneF32x2;
using R = F2;

constexpr int kM = 1024;
constexpr int kXBytes = 33 * 32 * 8;   // padded 32x32 transpose buffer, 8-byte elements
constexpr int kTabBytes = 2 * 1024 * 8; // T + TS
constexpr int kCtlBytes = 128;          // mbarriers + counters + TMEM base address

__device__ __forceinline__ R ld_stream_b64(const void *p)
{
    R r;
    asm volatile("ld.global.nc.L1::no_allocate.b64 %0, [%1];" : "=l"(r.v) : "l"(p));
    return r;
}
__device__ __forceinline__ int ld_stream_b32(const void *p)
{
    int r;
    asm volatile("ld.global.nc.L1::no_allocate.b32 %0, [%1];" : "=r"(r) : "l"(p));
    return r;
}
__device__ __forceinline__ float4 ld_nc_f4(const float4 *p)
{
    float4 r;
    asm volatile("ld.global.nc.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "l"(p));
    return r;
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

__device__ __forceinline__ unsigned long long l2_policy_evict_first()
{
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
// streamed output with an L2 evict_first hint: the written lines leave the L2 first instead of pushing the
// L2-prefetched traces out
__device__ __forceinline__ void st_global_b64_stream(void *p, R v, unsigned long long pol)
{
    asm volatile("st.global.L2::cache_hint.b64 [%0], %1, %2;" ::"l"(p), "l"(v.v), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_global_b64(void *p, R v)
{
    asm volatile("st.global.b64 [%0], %1;" ::"l"(p), "l"(v.v) : "memory");
}

// Outputs of one inverse transform: lane a, register b holds z[m = a + 32 b] of (theta, phi);
// sample index n = 2 m + parity. Both routines track the maximum of env^2 over b (ascending,
// strict >, so the lowest b wins ties).
//
// Even samples come out one whole inverse transform before the odd ones. Writing them straight to
// global memory would fill only half of every 32-byte sector, and the half-written sectors get
// evicted from L2 (ECC read-modify-write in DRAM: +35 % read, +13 % write traffic measured). So
// the even pass parks Re z (theta, phi) in this lane's tensor-memory columns and the odd pass
// stores (even, odd) pairs.
template <bool HAS_EF>
__device__ __forceinline__ void emit_even(const R (&zr)[32], const R (&zi)[32], uint32_t tpark, float &best, int &bb)
{
    static_for<0, 32>([&](auto bc) {
        constexpr int b = decltype(bc)::value;
        if (HAS_EF) tmem_st64(tpark + 2 * b, zr[b].v);
        R q = L::mul(zr[b], zr[b]);
        q = L::fma(zi[b], zi[b], q);
        float qt, qp;
        L::unpack(q, qt, qp);
        const float e2 = qt + qp;
        if (e2 > best) { best = e2; bb = b; }
    });
}

// Odd pass: lane l, row b fetches its parked even sample and stores the (even, odd) pair of theta
// at e_theta[2 (l + 32 b)] and of phi at e_phi[2 (l + 32 b)]: 8 bytes per lane, 256 contiguous
// bytes per instruction. The parked values come back in chunks of eight rows.
template <bool HAS_EF>
__device__ __forceinline__ void emit_odd(const R (&zr)[32], const R (&zi)[32], int lane, uint32_t tpark, float *ef,
                                         float &best, int &bb)
{
    static_for<0, 4>([&](auto cc) {
        constexpr int c = decltype(cc)::value;
        unsigned long long ev[8];
        if (HAS_EF) {
            static_for<0, 8>([&](auto jc) {
                constexpr int j = decltype(jc)::value;
                ev[j] = tmem_ld64(tpark + 2 * (8 * c + j));
            });
            tmem_wait_ld();
            static_for<0, 4>([&](auto jc) {
                constexpr int j = decltype(jc)::value;
                tmem_ld_dep(ev[2 * j], ev[2 * j + 1]);
            });
        }
        static_for<0, 8>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            constexpr int b = 8 * c + j;
            if (HAS_EF) {
                float ot, op, et, ep;
                L::unpack(zr[b], ot, op);
                R e; e.v = ev[j];
                L::unpack(e, et, ep);
                st_global_b64(ef + 2 * (lane + 32 * b), L::pack(et, ot));
                st_global_b64(ef + 2 * kM + 2 * (lane + 32 * b), L::pack(ep, op));
            }
            R q = L::mul(zr[b], zr[b]);
            q = L::fma(zi[b], zi[b], q);
            float qt, qp;
            L::unpack(q, qt, qp);
            const float e2 = qt + qp;
            if (e2 > best) { best = e2; bb = b; }
        });
    });
}

// ---- (even, odd) sample packing: the two halves of a packed register carry z[2m] and z[2m+1] of ONE polarisation
// (inputs E_p[k] and E_p[k] W_2048^-k share the transform's twiddles), the polarisations follow one another.
// Re z then leaves the transform as the (even, odd) pair an 8-byte store wants: no parking of samples, no register
// shuffles to pair them up; |z_theta|^2 of both samples waits in tensor memory for |z_phi|^2.
template <class G>
__device__ __forceinline__ void build_inverse_input_eo(R (&Zr)[32], R (&Zi)[32], const float2 *TS, int lane, uint32_t tstash_p)
{
    // tstash_p = stash + polarisation: columns 4 r + p (Re E_p) and 4 r + 2 + p (Im E_p) of band row r
    uint32_t er[G::kBandRows], ei[G::kBandRows];
    static_for<0, G::kBandRows>([&](auto rc) {
        constexpr int r = decltype(rc)::value;
        er[r] = tmem_ld32(tstash_p + 4 * r);
        ei[r] = tmem_ld32(tstash_p + 4 * r + 2);
    });
    tmem_wait_ld();
    static_for<0, 32>([&](auto kc) {
        constexpr int k2 = decltype(kc)::value;
        if constexpr (k2 < G::kLo || k2 > G::kHi) { Zr[brev5(k2)] = L::zero(); Zi[brev5(k2)] = L::zero(); }
        else {
            constexpr int r = k2 - G::kLo;
            tmem_ld_dep32(er[r], ei[r]);
            const float2 w = TS[lane + 32 * k2];
            const float sr = __uint_as_float(er[r]), si = __uint_as_float(ei[r]);
            // odd samples: (sr + i si)(wr - i wi)
            const float orr = fmaf(si, w.y, sr * w.x), oi = fmaf(-sr, w.y, si * w.x);
            Zr[brev5(k2)] = L::pack(sr, orr);
            Zi[brev5(k2)] = L::pack(si, oi);
        }
    });
}

// theta pass: store Re z_theta as (even, odd) pairs, park |z_theta|^2 of both samples
template <bool HAS_EF>
__device__ __forceinline__ void emit_theta(const R (&zr)[32], const R (&zi)[32], int lane, uint32_t tpark, float *ef, unsigned long long pol)
{
    static_for<0, 32>([&](auto bc) {
        constexpr int b = decltype(bc)::value;
        if (HAS_EF) st_global_b64_stream(ef + 2 * (lane + 32 * b), zr[b], pol);
        R q = L::mul(zr[b], zr[b]);
        q = L::fma(zi[b], zi[b], q);
        tmem_st64(tpark + 2 * b, q.v);
    });
}

// phi pass: store Re z_phi, env^2 = parked |z_theta|^2 + |z_phi|^2 for the even and the odd sample of every row,
// running (max, lowest row) per parity
template <bool HAS_EF>
__device__ __forceinline__ void emit_phi(const R (&zr)[32], const R (&zi)[32], int lane, uint32_t tpark, float *ef, unsigned long long pol,
                                         float &best0, int &b0, float &best1, int &b1)
{
    tmem_wait_st();
    static_for<0, 4>([&](auto cc) {
        constexpr int c = decltype(cc)::value;
        unsigned long long ev[8];
        static_for<0, 8>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            ev[j] = tmem_ld64(tpark + 2 * (8 * c + j));
        });
        tmem_wait_ld();
        static_for<0, 4>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            tmem_ld_dep(ev[2 * j], ev[2 * j + 1]);
        });
        static_for<0, 8>([&](auto jc) {
            constexpr int j = decltype(jc)::value;
            constexpr int b = 8 * c + j;
            if (HAS_EF) st_global_b64_stream(ef + 2 * kM + 2 * (lane + 32 * b), zr[b], pol);
            R q; q.v = ev[j];
            q = L::fma(zr[b], zr[b], q);
            q = L::fma(zi[b], zi[b], q);
            float e0, e1;
            L::unpack(q, e0, e1);
            if (e0 > best0) { best0 = e0; b0 = b; }
            if (e1 > best1) { best1 = e1; b1 = b; }
        });
    });
}

// Per-instantiation geometry: shared memory per warp, tensor-memory columns per warp, warps per CTA.
template <int K2LO, int K2HI>
struct W32Geom {
    static constexpr int kLo = K2LO, kHi = K2HI;
    // <10, 28> is used only for bands whose rows are exactly 10..28 (configs[1]); every other geometry serves any band
    // whose rows lie inside it, so its edge rows may be entirely out of band
    static constexpr bool kExact = K2LO == 10 && K2HI == 28;
    static constexpr int kBandRows = K2HI - K2LO + 1;
    // rows that hold some band bin's mirror 1024-k: row 31-r for lanes >= 1, row 32-r for lane 0
    static constexpr int kMirLo = 31 - K2HI;
    static constexpr int kMirHi = (32 - K2LO) > 31 ? 31 : (32 - K2LO);
    // rows of the forward spectrum published to shared memory: the band rows and their mirror rows
    static constexpr int kPubLo = kMirLo < K2LO ? kMirLo : K2LO;
    static constexpr int kPubHi = kMirHi > K2HI ? kMirHi : K2HI;
    static constexpr int kPubRows = kPubHi - kPubLo + 1;
    // one buffer per warp: the padded 32x32 transpose plane, reused for the published spectrum
    // (two planes of kPubRows x 32 packed values)
    static constexpr int kWarpBytes = kXBytes > kPubRows * 512 ? kXBytes : kPubRows * 512;
    // tensor-memory columns (32-bit, per lane): stash of E, 4 per band row, then the parked even samples
    static constexpr int kStashCols = 4 * kBandRows;
    static constexpr int kParkCol = kStashCols;
    static constexpr int kCols = kStashCols + 64;
    // warps of one scheduler share that scheduler's 32 TMEM lanes, so they split the 512 columns
    static constexpr int kWarps = 3 * kCols <= 512 ? 12 : 8;
    static constexpr int kColStride = 512 / (kWarps / 4);
    static_assert(kCols <= kColStride, "tensor-memory columns per warp");
};


// Input of one inverse transform, element k2 at position brev5(k2): E[k] (even samples) or
// E[k] W_2048^-k (ODD) on the band rows, zero elsewhere. E comes back from tensor memory.
template <class G, bool ODD>
__device__ __forceinline__ void build_inverse_input(R (&Zr)[32], R (&Zi)[32], const float2 *TS, int lane, uint32_t tstash)
{
    static_for<0, 32>([&](auto kc) {
        constexpr int k2 = decltype(kc)::value;
        if constexpr (k2 < G::kLo || k2 > G::kHi) { Zr[brev5(k2)] = L::zero(); Zi[brev5(k2)] = L::zero(); }
        else {
            Zr[brev5(k2)].v = tmem_ld64(tstash + 4 * (k2 - G::kLo));
            Zi[brev5(k2)].v = tmem_ld64(tstash + 4 * (k2 - G::kLo) + 2);
        }
    });
    tmem_wait_ld();
    static_for<G::kLo, G::kHi + 1>([&](auto kc) {
        constexpr int k2 = decltype(kc)::value;
        tmem_ld_dep(Zr[brev5(k2)].v, Zi[brev5(k2)].v);
        if (ODD) {
            const float2 w = TS[lane + 32 * k2];
            const R sr = Zr[brev5(k2)], si = Zi[brev5(k2)];
            // (sr + i si)(wr - i wi)
            R er = L::mul(sr, L::bc(w.x)); er = L::fma(si, L::bc(w.y), er);
            R ei = L::mul(si, L::bc(w.x)); ei = L::fma(sr, L::bc(-w.y), ei);
            Zr[brev5(k2)] = er; Zi[brev5(k2)] = ei;
        }
    });
}

} // namespace
} // namespace aera

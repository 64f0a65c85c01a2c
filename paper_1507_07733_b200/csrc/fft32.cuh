// Register-resident 32-point FFT and packed-lane arithmetic for the warp kernels.
//
// Lane types ("two transforms for the price of one issue slot"):
//   LaneF32x2 : one 64-bit register pair holding two independent fp32 values, driven by the sm_100
//               packed instructions fma/add/sub/mul.rn.f32x2 (SASS FFMA2/FADD2/FMUL2). Two FFTs with
//               identical twiddles ride in the two halves: measured 2 warp-instr/clk/SM = the same 128
//               lane-FMAs/clk as scalar FFMA but half the issue slots. Twiddles are scalars: ptxas
//               folds mov.b64 {w,w} into the .F32 broadcast operand (or an immediate) and folds
//               negations into operand modifiers, so they cost no registers or instructions.
//   LaneF64   : plain double (one transform), same code.
//
// fft32<L>(re, im): in-place radix-2 decimation-in-time, input element j at position brev5(j),
// output in natural order, forward sign exp(-2 pi i jk/32), unnormalised. The inverse transform is
// the same routine called with the arrays swapped: IFFT(x) = swap(FFT(swap(x))) (un-normalised).
// Every butterfly is the FMA form  u = a + W b (4 FMA), v = 2a - u (2 FMA): 6 ops instead of 8;
// W = 1 and W = -i butterflies are 4 adds; W = (+-1 - i)/sqrt2 are 2 adds + 4 FMA.
#pragma once
#include <cstdint>
#include <type_traits>

namespace aera {

typedef unsigned long long u64_t;

struct F2 { u64_t v; };

struct LaneF32x2 {
    using R = F2;
    using S = float;
    static __device__ __forceinline__ R pack(float lo, float hi) { R r; asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi)); return r; }
    static __device__ __forceinline__ void unpack(R a, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); }
    static __device__ __forceinline__ R bc(S s) { return pack(s, s); }
    static __device__ __forceinline__ R zero() { R r; r.v = 0ull; return r; }
    static __device__ __forceinline__ R neg(R a) { float x, y; unpack(a, x, y); return pack(-x, -y); }
    static __device__ __forceinline__ R add(R a, R b) { R r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
    static __device__ __forceinline__ R sub(R a, R b) { R r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
    static __device__ __forceinline__ R mul(R a, R b) { R r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v)); return r; }
    static __device__ __forceinline__ R fma(R a, R b, R c) { R r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return r; }
};

struct LaneF64 {
    using R = double;
    using S = double;
    static __device__ __forceinline__ R bc(S s) { return s; }
    static __device__ __forceinline__ R zero() { return 0.0; }
    static __device__ __forceinline__ R neg(R a) { return -a; }
    static __device__ __forceinline__ R add(R a, R b) { return __dadd_rn(a, b); }
    static __device__ __forceinline__ R sub(R a, R b) { return __dsub_rn(a, b); }
    static __device__ __forceinline__ R mul(R a, R b) { return __dmul_rn(a, b); }
    static __device__ __forceinline__ R fma(R a, R b, R c) { return __fma_rn(a, b, c); }
};

struct LaneF32 {   // plain float lanes (one transform), same code
    using R = float;
    using S = float;
    static __device__ __forceinline__ R bc(S s) { return s; }
    static __device__ __forceinline__ R zero() { return 0.0f; }
    static __device__ __forceinline__ R neg(R a) { return -a; }
    static __device__ __forceinline__ R add(R a, R b) { return __fadd_rn(a, b); }
    static __device__ __forceinline__ R sub(R a, R b) { return __fsub_rn(a, b); }
    static __device__ __forceinline__ R mul(R a, R b) { return __fmul_rn(a, b); }
    static __device__ __forceinline__ R fma(R a, R b, R c) { return __fmaf_rn(a, b, c); }
};

template <int I> using IC = std::integral_constant<int, I>;
template <int B, int E, class F>
__device__ __forceinline__ void static_for(F &&f)
{
    if constexpr (B < E) {
        f(IC<B>{});
        static_for<B + 1, E>(f);
    }
}

__host__ __device__ constexpr int brev5(int j)
{
    return ((j & 1) << 4) | ((j & 2) << 2) | (j & 4) | ((j & 8) >> 2) | ((j & 16) >> 4);
}

// cos/sin(2 pi i / 32), i = 0..15
__device__ constexpr double kCos32[16] = {
    1.0, 0.98078528040323044913, 0.92387953251128675613, 0.83146961230254523708,
    0.70710678118654752440, 0.55557023301960222474, 0.38268343236508977173, 0.19509032201612826785,
    0.0, -0.19509032201612826785, -0.38268343236508977173, -0.55557023301960222474,
    -0.70710678118654752440, -0.83146961230254523708, -0.92387953251128675613, -0.98078528040323044913};
__device__ constexpr double kSin32[16] = {
    0.0, 0.19509032201612826785, 0.38268343236508977173, 0.55557023301960222474,
    0.70710678118654752440, 0.83146961230254523708, 0.92387953251128675613, 0.98078528040323044913,
    1.0, 0.98078528040323044913, 0.92387953251128675613, 0.83146961230254523708,
    0.70710678118654752440, 0.55557023301960222474, 0.38268343236508977173, 0.19509032201612826785};

// (a, b) <- (a + W b, a - W b), W = exp(-2 pi i IDX/32)
template <class L, int IDX>
__device__ __forceinline__ void butterfly(typename L::R &ar, typename L::R &ai, typename L::R &br, typename L::R &bi)
{
    using R = typename L::R;
    using S = typename L::S;
    if constexpr (IDX == 0) {
        R ur = L::add(ar, br), ui = L::add(ai, bi);
        br = L::sub(ar, br); bi = L::sub(ai, bi);
        ar = ur; ai = ui;
    } else if constexpr (IDX == 8) { // W = -i : W b = (bi, -br)
        R ur = L::add(ar, bi), ui = L::sub(ai, br);
        R vr = L::sub(ar, bi), vi = L::add(ai, br);
        ar = ur; ai = ui; br = vr; bi = vi;
    } else if constexpr (IDX == 4) { // W = h(1 - i) : W b = h((br + bi), (bi - br))
        const R h = L::bc((S)0.70710678118654752440), nh = L::bc((S)-0.70710678118654752440);
        R s1 = L::add(br, bi), s2 = L::sub(bi, br);
        R ur = L::fma(s1, h, ar), ui = L::fma(s2, h, ai);
        br = L::fma(s1, nh, ar); bi = L::fma(s2, nh, ai);
        ar = ur; ai = ui;
    } else if constexpr (IDX == 12) { // W = h(-1 - i) : W b = h((bi - br), -(br + bi))
        const R h = L::bc((S)0.70710678118654752440), nh = L::bc((S)-0.70710678118654752440);
        R s1 = L::sub(bi, br), s2 = L::add(br, bi);
        R ur = L::fma(s1, h, ar), ui = L::fma(s2, nh, ai);
        br = L::fma(s1, nh, ar); bi = L::fma(s2, h, ai);
        ar = ur; ai = ui;
    } else { // W = c - i s : W b = (c br + s bi, c bi - s br)
        const R c = L::bc((S)kCos32[IDX]), s = L::bc((S)kSin32[IDX]), ns = L::bc((S)(-kSin32[IDX])), two = L::bc((S)2.0);
        R ur = L::fma(br, c, ar);
        ur = L::fma(bi, s, ur);
        R ui = L::fma(bi, c, ai);
        ui = L::fma(br, ns, ui);
        br = L::fma(ar, two, L::neg(ur));
        bi = L::fma(ai, two, L::neg(ui));
        ar = ur; ai = ui;
    }
}

template <class L>
__device__ __forceinline__ void fft32(typename L::R (&re)[32], typename L::R (&im)[32])
{
    static_for<0, 5>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        constexpr int half = 1 << s;
        static_for<0, 16>([&](auto bc) {
            constexpr int b = decltype(bc)::value;      // butterfly number 0..15
            constexpr int j = b & (half - 1);
            constexpr int i0 = ((b - j) << 1) + j;
            constexpr int i1 = i0 + half;
            constexpr int idx = j * (16 >> s);
            butterfly<L, idx>(re[i0], im[i0], re[i1], im[i1]);
        });
    });
}

// The same transform when only the input ELEMENTS NZLO..NZHI are non-zero (the first pass of an inverse transform whose
// spectrum is confined to the band rows): in stage 0, which pairs element e with e + 16, a butterfly with one zero
// input is a copy (b = 0) or a copy and a negation (a = 0; ptxas folds the negation into the consumers' operand
// modifiers), with two zero inputs nothing. The zero elements are never read, so the caller need not store them.
// (From stage 1 on every value is non-zero for the bands of interest and the stages are the plain ones.)
template <class L, int NZLO, int NZHI>
__device__ __forceinline__ void fft32_pruned(typename L::R (&re)[32], typename L::R (&im)[32])
{
    static_for<0, 16>([&](auto bc) {
        constexpr int b = decltype(bc)::value;
        constexpr int i0 = 2 * b, i1 = i0 + 1;
        constexpr int e0 = brev5(i0), e1 = brev5(i1);        // element indices: e1 = e0 + 16
        constexpr bool za = e0 < NZLO || e0 > NZHI, zb = e1 < NZLO || e1 > NZHI;
        if constexpr (za && zb) { re[i0] = L::zero(); im[i0] = L::zero(); re[i1] = L::zero(); im[i1] = L::zero(); }
        else if constexpr (zb) { re[i1] = re[i0]; im[i1] = im[i0]; }
        else if constexpr (za) { re[i0] = re[i1]; im[i0] = im[i1]; re[i1] = L::neg(re[i1]); im[i1] = L::neg(im[i1]); }
        else butterfly<L, 0>(re[i0], im[i0], re[i1], im[i1]);
    });
    static_for<1, 5>([&](auto sc) {
        constexpr int s = decltype(sc)::value;
        constexpr int half = 1 << s;
        static_for<0, 16>([&](auto bc) {
            constexpr int b = decltype(bc)::value;
            constexpr int j = b & (half - 1);
            constexpr int i0 = ((b - j) << 1) + j;
            constexpr int i1 = i0 + half;
            constexpr int idx = j * (16 >> s);
            butterfly<L, idx>(re[i0], im[i0], re[i1], im[i1]);
        });
    });
}

} // namespace aera

// Warp-per-station fused unfolding kernel for N = 2048 fp32 (BASELINE configs[1], the headline).
//
// One warp owns one station at a time. Every transform is a 1024-point complex FFT done as
// 32 x 32: each lane runs a 32-point FFT in registers (fft32.cuh), the warp transposes through
// shared memory once, each lane runs a second 32-point FFT. Two transforms ride in the two halves
// of the packed f32x2 lanes:
//
//   a1/a2 forward : g_r[m] = v0[2m+r] + i v1[2m+r], r = 0,1 in the two lanes. An 8-byte load of
//                   channel 0 IS the packed real part, of channel 1 the packed imaginary part.
//                   G_r = FFT_1024(g_r).  With the mirror bin 1024-k (one exchange through shared
//                   memory) the four real polyphase spectra separate, and
//                   2 V_c[k] = F'_c0[k] + W_2048^k F'_c1[k]   (k < 1024 covers the whole band).
//   a4 solve      : (E_theta, E_phi)[k] = Minv[event][k] (V_0, V_1)[k]; Minv = (1/N) H^-1 comes from
//                   pattern.cu once per event as two zero-padded planes (MINV_PACKED_PAD), so band-edge rows
//                   multiply by zero instead of clamping and selecting. E goes to tensor memory.
//   a5 inverse    : the analytic spectrum is zero above N/2, so (z_p[2m], z_p[2m+1]) = IFFT_1024 of
//                   (E_p[k], E_p[k] W_2048^{-k}): ONE packed transform per polarisation whose two lanes
//                   are the even and the odd samples (theta first, then phi), instead of two 2048-point
//                   ones. The inverse is the forward routine with the re/im arrays swapped.
//   a6 outputs    : Re z_p leaves the transform as the (even, odd) pair of an 8-byte store, straight from
//                   registers. The theta pass parks |z_theta|^2 of both samples in tensor memory; the phi
//                   pass adds |z_phi|^2 and keeps a running (max, lowest row) per lane and parity; the
//                   warp argmax is two integer REDUX reductions (max of the float bits, then min index).
//
// Work distribution: CTA b owns the contiguous unit range [b n/G, (b+1) n/G); its twelve warps stride
// through it. All stations of an event share Minv (one direction per event), so the
// CTA keeps the current and the next event's Minv (20 KB each at configs[1]) in shared memory:
// TMA bulk copies (cp.async.bulk + mbarrier) fill a two-slot ring; the last warp to leave event e
// (shared-memory counter) issues the copy of event e+2 into the slot it vacates.
//
// HBM traffic per station: 16 KB read once (L2-prefetched one station ahead with
// cp.async.bulk.prefetch.L2), 16 KB + 8 B written once, as (even, odd) sample pairs: 8 bytes per
// lane, 256 contiguous bytes per store instruction, every 32-byte sector written once and in full,
// with an L2 evict_first hint so the written lines do not push the prefetched traces out.
//
// Lane-private scratch lives in tensor memory (tmem.cuh), not in shared memory: the in-band
// spectrum E (read once per polarisation) and the parked |z_theta|^2. That leaves one 10 KB
// transpose / mirror-exchange buffer per warp in shared memory, so twelve warps (168 registers each)
// fit on an SM instead of eight: three warps per scheduler hide each other's shared-memory and
// global-memory latencies.
//
// The in-band rows (bins k = lane + 32 row) are template parameters, so every per-row decision is
// made at compile time; <10, 28> is configs[1] (k = 342..910), <0, 31> serves any other band.
#include "w32_common.cuh"

namespace aera {
namespace {

constexpr int kSolveUnroll = 1;   // band rows of separate_solve in flight together (2 and 4 measured slower)

struct W32Params {
    const void *traces;    // float [n_units][2][2048], or int16 ADC counts of the same shape (IN16)
    const int32_t *pattern_id; // [n_stations] antenna type per station, or nullptr (one table)
    size_t minv_pattern_stride; // float4 elements between the Minv slabs of consecutive tables
    float *efield;
    float *amp;
    int32_t *idx;
    const float4 *minv;   // [n_events] { A[K + 64], B[K + 64] } float4, see MINV_PACKED_PAD
    float4 *spectra;      // [n_units][band rows][32] {2V0.re, 2V0.im, 2V1.re, 2V1.im}: written (SPEC 1) or read (SPEC 2)
    const float2 *tw1024; // W_1024^m
    const float2 *twN;    // W_2048^m
    long n_units;
    int n_stations;
    int k_lo, k_hi, K;
};

// One band row per iteration: row k2 = kLo + r holds bin k = lane + 32 k2 of the packed forward
// spectrum G_r (r = 0, 1 in the two halves). Separates the channels with the mirror bin 1024-k,
// folds the two polyphase halves (2 V_c = F'_c0 + W_2048^k F'_c1), applies Minv (a4) and leaves
// (E_theta, E_phi) packed as (re, im) in tensor-memory columns 4r .. 4r+3 of this lane.
// SPEC = 1 also stores 2 V_c of the band rows (direction-independent: later iterations of the reconstruction loop
// start from them, SPEC = 2, and skip the trace read and the forward transform).
template <class G, bool MINV_SMEM, int SPEC>
__device__ __forceinline__ void separate_solve(const R *QA, const R *QB, const float2 *TS, const float4 *MA,
                                               const float4 *MB, int k_lo, int k_hi, int lane, uint32_t tstash, float4 *sp)
{
    // partner bin 1024-k lives in lane (32-lane)&31, row 31-k2 (row 32-k2 for lane 0)
    // (k = 0, whose partner row would be 32, is never in band: k_lo >= 1)
    int own = (G::kLo - G::kPubLo) * 32 + lane;
    int par = (31 - G::kLo + (lane == 0 ? 1 : 0) - G::kPubLo) * 32 + ((32 - lane) & 31);
    int k = lane + 32 * G::kLo;
#pragma unroll (kSolveUnroll)
    for (int r = 0; r < G::kBandRows; ++r, own += 32, par -= 32, k += 32) {
        // branch-free: rows at the band edges read a clamped Minv entry and select zero afterwards, so the
        // loads of neighbouring rows are independent and the unrolled iterations overlap their latencies
        // rows of a band-specific instantiation reach at most 31 bins beyond the band: Minv is zero-padded there
        // (MINV_PACKED_PAD), so E = 0 comes out of the arithmetic; the any-band instantiation clamps and selects
        constexpr bool kAnyBand = !G::kExact;   // instantiation rows are a superset of the band's rows
        const bool inband = !kAnyBand || (k >= k_lo && k <= k_hi);
        int j = k - k_lo;
        if (kAnyBand) j = j < 0 ? 0 : (j > k_hi - k_lo ? k_hi - k_lo : j);
        // (lane 0 of row 0 would look for its mirror in row 32: k = 0 is never in band, keep the read inside the buffer)
        const int pc = (G::kLo == 0 && par > G::kPubRows * 32 - 1) ? G::kPubRows * 32 - 1 : par;
        const R ar = QA[own], ai = QB[own], pr = QA[pc], pi = QB[pc];
        const float2 w = TS[k]; // W_2048^k = (wr, wi)
        const float4 m0 = MINV_SMEM ? MA[j] : ld_nc_f4(MA + j);
        const float4 m1 = MINV_SMEM ? MB[j] : ld_nc_f4(MB + j);
        // F'_0 = G + conj(Gm) = 2 FFT(v0 polyphase r), F'_1 = -i (G - conj(Gm)) = 2 FFT(v1 polyphase r)
        const R f0r = L::add(ar, pr), f0i = L::sub(ai, pi);
        const R f1r = L::add(ai, pi), f1i = L::sub(pr, ar);
        float f0r0, f0r1, f0i0, f0i1, f1r0, f1r1, f1i0, f1i1;
        L::unpack(f0r, f0r0, f0r1); L::unpack(f0i, f0i0, f0i1);
        L::unpack(f1r, f1r0, f1r1); L::unpack(f1i, f1i0, f1i1);
        float v0r = fmaf(w.x, f0r1, f0r0); v0r = fmaf(-w.y, f0i1, v0r);
        float v0i = fmaf(w.x, f0i1, f0i0); v0i = fmaf(w.y, f0r1, v0i);
        float v1r = fmaf(w.x, f1r1, f1r0); v1r = fmaf(-w.y, f1i1, v1r);
        float v1i = fmaf(w.x, f1i1, f1i0); v1i = fmaf(w.y, f1r1, v1i);
        if (kAnyBand && !inband) { v0r = 0.f; v0i = 0.f; v1r = 0.f; v1i = 0.f; }
        const R Ma = L::pack(m0.x, m0.y), Mb = L::pack(m0.z, m0.w), Mc = L::pack(m1.x, m1.y), Md = L::pack(m1.z, m1.w);
        R er = L::mul(Ma, L::bc(v0r)); er = L::fma(Mb, L::bc(-v0i), er);
        er = L::fma(Mc, L::bc(v1r), er); er = L::fma(Md, L::bc(-v1i), er);
        R ei = L::mul(Ma, L::bc(v0i)); ei = L::fma(Mb, L::bc(v0r), ei);
        ei = L::fma(Mc, L::bc(v1i), ei); ei = L::fma(Md, L::bc(v1r), ei);
        if (SPEC == 1) sp[r * 32] = make_float4(v0r, v0i, v1r, v1i);
        tmem_st64(tstash + 4 * r, er.v);
        tmem_st64(tstash + 4 * r + 2, ei.v);
    }
}

// SPEC = 2: a4 straight from the stored 2 V_c of this station (zero outside the band).
// The rows are first copied to the warp's shared-memory buffer with independent loads (one latency, not one
// per row of the rolled loop).
template <class G, bool MINV_SMEM>
__device__ __forceinline__ void solve_from_spectra(const float4 *sp, float4 *XV, const float4 *MA, const float4 *MB, int k_lo,
                                                   int k_hi, int lane, uint32_t tstash)
{
    static_assert(G::kBandRows * 512 <= G::kWarpBytes, "band rows fit the warp buffer");
    {
        float4 tmp[G::kBandRows];
        static_for<0, G::kBandRows>([&](auto rc) { constexpr int r = decltype(rc)::value; tmp[r] = ld_nc_f4(sp + r * 32); });
        static_for<0, G::kBandRows>([&](auto rc) { constexpr int r = decltype(rc)::value; XV[r * 32 + lane] = tmp[r]; });
    }
    __syncwarp();
    int k = lane + 32 * G::kLo;
#pragma unroll 1
    for (int r = 0; r < G::kBandRows; ++r, k += 32) {
        R er = L::zero(), ei = L::zero();
        if (k >= k_lo && k <= k_hi) {
            const float4 v = XV[r * 32 + lane];
            const float4 m0 = MINV_SMEM ? MA[k - k_lo] : ld_nc_f4(MA + (k - k_lo));
            const float4 m1 = MINV_SMEM ? MB[k - k_lo] : ld_nc_f4(MB + (k - k_lo));
            const R Ma = L::pack(m0.x, m0.y), Mb = L::pack(m0.z, m0.w), Mc = L::pack(m1.x, m1.y), Md = L::pack(m1.z, m1.w);
            er = L::mul(Ma, L::bc(v.x)); er = L::fma(Mb, L::bc(-v.y), er);
            er = L::fma(Mc, L::bc(v.z), er); er = L::fma(Md, L::bc(-v.w), er);
            ei = L::mul(Ma, L::bc(v.y)); ei = L::fma(Mb, L::bc(v.x), ei);
            ei = L::fma(Mc, L::bc(v.w), ei); ei = L::fma(Md, L::bc(v.z), ei);
        }
        tmem_st64(tstash + 4 * r, er.v);
        tmem_st64(tstash + 4 * r + 2, ei.v);
    }
}

template <int K2LO, int K2HI, bool HAS_EF, bool MINV_SMEM, int SPEC, bool IN16>
__global__ void __launch_bounds__(W32Geom<K2LO, K2HI>::kWarps * 32, 1)
unfold_w32_kernel(W32Params p)
{
    using G = W32Geom<K2LO, K2HI>;
    constexpr int kWarps = G::kWarps;
    extern __shared__ __align__(128) unsigned char smem[];
    float2 *T = reinterpret_cast<float2 *>(smem);               // [32][32] pass twiddles
    float2 *TS = T + 1024;                                       // [1024] W_2048^k
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + kTabBytes);     // [2] Minv slot filled
    int *done = reinterpret_cast<int *>(smem + kTabBytes + 16);          // [2] warps finished with the slot
    uint32_t *tmem_base = reinterpret_cast<uint32_t *>(smem + kTabBytes + 32);
    const int KP = p.K + 2 * kMinvPad;                          // entries per padded Minv plane
    const uint32_t minv_bytes = (uint32_t)KP * 32u;
    const uint32_t slot_bytes = MINV_SMEM ? ((minv_bytes + 127u) & ~127u) : 0u;
    unsigned char *mslot = smem + kTabBytes + kCtlBytes;
    // warp index through a shuffle: provably warp-uniform, so everything derived from it is too
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    unsigned char *wbase = mslot + 2 * (size_t)slot_bytes + (size_t)warp * G::kWarpBytes;
    R *X = reinterpret_cast<R *>(wbase);                         // transpose buffer
    R *QA = X;                                                   // published forward spectrum, real plane
    R *QB = X + G::kPubRows * 32;                                // ... imaginary plane

    const long S = p.n_stations;
    const long u0 = p.n_units * (long)blockIdx.x / (long)gridDim.x;
    const long u1 = p.n_units * ((long)blockIdx.x + 1) / (long)gridDim.x;
    // (no early exit: every CTA allocates and frees tensor memory; an empty range skips the loops)
    const long e0 = u0 / S, e1 = u1 > u0 ? (u1 - 1) / S : e0 - 1;

    if (warp == 0) tmem_alloc_all(tmem_base);
    if (MINV_SMEM && threadIdx.x == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        done[0] = 0; done[1] = 0;
        for (int s = 0; s < 2 && e0 + s <= e1; ++s) {
            mbar_expect_tx(&full[s], minv_bytes);
            tma_bulk_g2s(mslot + (size_t)s * slot_bytes, p.minv + (size_t)(e0 + s) * KP * 2, minv_bytes, &full[s]);
        }
    }
    for (int i = threadIdx.x; i < 1024; i += blockDim.x) {
        const int k1 = i >> 5, t = i & 31;
        T[i] = p.tw1024[(k1 * t) & 1023];
        TS[i] = p.twN[i];
    }
    tmem_fence_before_sync();
    __syncthreads();
    tmem_fence_after_sync();
    const uint32_t tbase = *tmem_base;
    const uint32_t tstash = tmem_addr(tbase, warp, (warp >> 2) * G::kColStride);
    const uint32_t tpark = tstash + G::kParkCol;
    const unsigned long long pol_first = l2_policy_evict_first();

#pragma unroll 1
    for (long e = e0; e <= e1; ++e) {
        const int slot = (int)((e - e0) & 1);
        const uint32_t parity = (uint32_t)(((e - e0) >> 1) & 1);
        const long lo = u0 > e * S ? u0 : e * S;
        const long hi = u1 < (e + 1) * S ? u1 : (e + 1) * S;
        const long first = lo + (((long)warp - (lo - u0)) % kWarps + kWarps) % kWarps;
        const float4 *MA = MINV_SMEM ? reinterpret_cast<const float4 *>(mslot + (size_t)slot * slot_bytes)
                                     : p.minv + (size_t)e * KP * 2;
        bool minv_ready = !MINV_SMEM;

#pragma unroll 1
        for (long u = first; u < hi; u += kWarps) {
            const float *v = static_cast<const float *>(p.traces) + (size_t)u * 4 * kM;
            const int16_t *v16 = static_cast<const int16_t *>(p.traces) + (size_t)u * 4 * kM;
            // several tables resident: this station's antenna type selects the Minv slab (read through L1/L2)
            const float4 *MAu = ((MINV_SMEM || p.pattern_id == nullptr) ? MA : MA + (size_t)p.pattern_id[u - e * S] * p.minv_pattern_stride) + kMinvPad;
            const float4 *MBu = MAu + KP;
            float *ef = HAS_EF ? p.efield + (size_t)u * 4 * kM : nullptr;
            float4 *sp = SPEC != 0 ? p.spectra + (size_t)u * G::kBandRows * 32 + lane : nullptr;
            if (lane == 0 && u + kWarps < u1) {          // this warp's next station, one ahead (two ahead measured no better)
                if (SPEC != 2 && IN16) prefetch_l2_bulk(v16 + (size_t)kWarps * 4 * kM, 4 * kM * sizeof(int16_t));
                else if (SPEC != 2) prefetch_l2_bulk(v + (size_t)kWarps * 4 * kM, 4 * kM * sizeof(float));
                else prefetch_l2_bulk(p.spectra + (size_t)(u + kWarps) * G::kBandRows * 32, G::kBandRows * 32 * sizeof(float4));
            }

            R A[32], B[32];
            if constexpr (SPEC != 2) {
                // ---- a1: the station's two traces, read once, straight into FFT input order
                static_for<0, 32>([&](auto jc) {
                    constexpr int j = decltype(jc)::value;
                    if (IN16) { // two ADC counts per 32-bit word: (v[2m], v[2m+1]); the counts-to-volts factors are in Minv
                        const int a = ld_stream_b32(v16 + 2 * (lane + 32 * j)), b = ld_stream_b32(v16 + 2 * kM + 2 * (lane + 32 * j));
                        A[brev5(j)] = L::pack((float)(short)(a & 0xffff), (float)(a >> 16));
                        B[brev5(j)] = L::pack((float)(short)(b & 0xffff), (float)(b >> 16));
                        return;
                    }
                    A[brev5(j)] = ld_stream_b64(v + 2 * (lane + 32 * j));            // (v0[2m], v0[2m+1])
                    B[brev5(j)] = ld_stream_b64(v + 2 * kM + 2 * (lane + 32 * j));   // (v1[2m], v1[2m+1])
                });
            } else {
                // ---- the forward spectrum of this station was stored by an earlier call: a4 straight away
                if (!minv_ready) { mbar_wait(&full[slot], parity); minv_ready = true; }
                solve_from_spectra<G, MINV_SMEM>(sp, reinterpret_cast<float4 *>(X), MAu, MBu, p.k_lo, p.k_hi, lane, tstash);
                __syncwarp(); // the buffer becomes a transpose plane again
                tmem_wait_st();
                build_inverse_input_eo<G>(B, A, TS, lane, tstash);
            }

            // ---- three 1024-point transforms through ONE copy of the FFT code (the instruction
            // stream of a fully unrolled station is ~90 KB, far beyond the instruction caches; with
            // twelve warps at different places in it, instruction fetch was the first limiter):
            //   t = 0 forward (A = Re, B = Im); t = 1, 2 inverse, which is the forward routine with
            //   the roles swapped (A = Im, B = Re).
            float best0 = -1.0f, best1 = -1.0f; int b0 = 0, b1 = 0;
            // (Loops are written so that each exit leaves straight from the FFT: a join of the
            // "continue" and "exit" paths would cost a register shuffle on every pass.)
            int t = SPEC == 2 ? 1 : 0;
#pragma unroll 1
            for (;;) {
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
                if (t == 2) break;
                if (SPEC != 2 && t == 0) {
                    // ---- a2 done: publish the band rows and the rows that are somebody's bin 1024-k
                    static_for<G::kPubLo, G::kPubHi + 1>([&](auto rc) {
                        constexpr int r = decltype(rc)::value;
                        QA[(r - G::kPubLo) * 32 + lane] = A[r];
                        QB[(r - G::kPubLo) * 32 + lane] = B[r];
                    });
                    __syncwarp();
                    if (!minv_ready) { mbar_wait(&full[slot], parity); minv_ready = true; }
                    // ---- separate channels, fold the two polyphase halves, a4: E = Minv V, one band
                    // row per iteration (a rolled loop: 40 instructions instead of 19 x 45), E goes to
                    // this lane's tensor-memory columns and is read back once per polarisation
                    separate_solve<G, MINV_SMEM, SPEC>(QA, QB, TS, MAu, MBu, p.k_lo, p.k_hi, lane, tstash, sp);
                    __syncwarp(); // all reads of the published rows done before the buffer is a transpose plane again
                    tmem_wait_st();
                } else
                    emit_theta<HAS_EF>(B, A, lane, tpark, ef, pol_first);
                // ---- a5 (one copy of the code for both polarisations; the registers are dead at this join):
                // (z[2m], z[2m+1]) = IFFT_1024 of (E_p, E_p W_2048^-k), p = theta after t = 0, phi after t = 1;
                // inverse roles, A = Im, B = Re
                build_inverse_input_eo<G>(B, A, TS, lane, tstash + (uint32_t)t);
                ++t;
            }
            emit_phi<HAS_EF>(B, A, lane, tpark, ef, pol_first, best0, b0, best1, b1);

            // ---- a6: lane result (lowest index on ties), then warp argmax with the same rule
            float best = best0; int bi = 2 * (lane + 32 * b0);
            {
                const int n1 = 2 * (lane + 32 * b1) + 1;
                if (best1 > best || (best1 == best && n1 < bi)) { best = best1; bi = n1; }
            }
            // env^2 >= 0, so the float order is the order of the bit patterns: two warp-wide integer reductions
            // (REDUX) instead of five shuffle stages: the maximum, then the lowest index among the lanes that hold it
            {
                const unsigned bmax = __reduce_max_sync(0xffffffffu, __float_as_uint(best));
                bi = (int)__reduce_min_sync(0xffffffffu, __float_as_uint(best) == bmax ? (unsigned)bi : 0xffffffffu);
                best = __uint_as_float(bmax);
            }
            if (lane == 0) { p.amp[u] = sqrtf(best); p.idx[u] = bi; }
        }

        if (MINV_SMEM) {
            // Leave event e. Every warp passes through here exactly once per event, and only after
            // it saw the slot full, so the counter cannot run ahead of the copy it guards.
            if (!minv_ready) mbar_wait(&full[slot], parity);
            __syncwarp();
            if (lane == 0) {
                __threadfence_block();
                const int old = atomicAdd(&done[slot], 1);
                if (old == kWarps - 1) {
                    done[slot] = 0;
                    __threadfence_block();
                    if (e + 2 <= e1) {
                        fence_proxy_async_smem();
                        mbar_expect_tx(&full[slot], minv_bytes);
                        tma_bulk_g2s(mslot + (size_t)slot * slot_bytes, p.minv + (size_t)(e + 2) * KP * 2, minv_bytes, &full[slot]);
                    }
                }
            }
        }
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_free_all(tbase);
}

template <int K2LO, int K2HI, bool MINV_SMEM>
size_t w32_smem_bytes(int K)
{
    using G = W32Geom<K2LO, K2HI>;
    const size_t slot = MINV_SMEM ? (((size_t)(K + 2 * kMinvPad) * 32 + 127) & ~(size_t)127) : 0;
    return (size_t)kTabBytes + kCtlBytes + 2 * slot + (size_t)G::kWarps * G::kWarpBytes;
}

template <int K2LO, int K2HI, bool HAS_EF, bool MINV_SMEM, int SPEC, bool IN16 = false>
cudaError_t launch_inst(const W32Params &q, cudaStream_t s)
{
    using G = W32Geom<K2LO, K2HI>;
    const size_t smem = w32_smem_bytes<K2LO, K2HI, MINV_SMEM>(q.K);
    auto kern = unfold_w32_kernel<K2LO, K2HI, HAS_EF, MINV_SMEM, SPEC, IN16>;
    AERA_ENSURE_DYN_SMEM(kern, smem);
    long grid = (q.n_units + G::kWarps - 1) / G::kWarps;
    if (grid > sm_count()) grid = sm_count();
    kern<<<(unsigned)grid, G::kWarps * 32, smem, s>>>(q);
    return cudaGetLastError();
}

} // namespace

bool w32_supported(int dtype, const PlanDev &p)
{
    return dtype == AERA_F32 && p.N == 2 * kM && p.k_hi < kM && p.k_lo >= 1;
}

// Row geometries instantiated: <10, 28> exactly configs[1]'s rows (30-80 MHz at fs = 180 MHz); <6, 28> any band inside
// bins 192..927 (30-80 MHz at sampling rates of 180-250 MHz: still twelve warps and the per-event Minv ring);
// <0, 31> everything else (eight warps, Minv through L1/L2).
static int w32_geom(const PlanDev &p)
{
    const int lo = p.k_lo >> 5, hi = p.k_hi >> 5;
    if (lo == 10 && hi == 28) return 0;
    if (lo >= 6 && hi <= 28) return 1;
    return 2;
}

size_t w32_spectra_bytes(const PlanDev &p, long n_units)
{
    const int g = w32_geom(p);
    const int rows = g == 0 ? W32Geom<10, 28>::kBandRows : (g == 1 ? W32Geom<6, 28>::kBandRows : 32);
    return (size_t)n_units * rows * 32 * sizeof(float4);
}

namespace {
// MINV_RING: the geometry stages Minv per event in shared memory (unless several tables are resident)
template <int K2LO, int K2HI, bool MINV_RING>
cudaError_t launch_geom(const W32Params &q, cudaStream_t s, bool ef, bool i16, bool multi, int spec)
{
    if (i16) return ef ? launch_inst<K2LO, K2HI, true, MINV_RING, 0, true>(q, s) : launch_inst<K2LO, K2HI, false, MINV_RING, 0, true>(q, s);
    if (multi) return ef ? launch_inst<K2LO, K2HI, true, false, 0>(q, s) : launch_inst<K2LO, K2HI, false, false, 0>(q, s);
    if (spec == 1) return ef ? launch_inst<K2LO, K2HI, true, MINV_RING, 1>(q, s) : launch_inst<K2LO, K2HI, false, MINV_RING, 1>(q, s);
    if (spec == 2) return ef ? launch_inst<K2LO, K2HI, true, MINV_RING, 2>(q, s) : launch_inst<K2LO, K2HI, false, MINV_RING, 2>(q, s);
    return ef ? launch_inst<K2LO, K2HI, true, MINV_RING, 0>(q, s) : launch_inst<K2LO, K2HI, false, MINV_RING, 0>(q, s);
}
} // namespace

cudaError_t launch_unfold_w32(const PlanDev &p, long n_events, int n_stations, const void *traces, void *efield,
                              void *amp, int32_t *idx, const void *minv, cudaStream_t s, void *spectra, int spec_mode,
                              const UnfoldExt &x)
{
    const long n_units = n_events * (long)n_stations;
    if (n_units <= 0) return cudaSuccess;
    ProfScope prof(KID_UNFOLD, s);
    W32Params q;
    q.traces = traces; q.efield = (float *)efield; q.amp = (float *)amp; q.idx = idx;
    q.pattern_id = x.pattern_id; q.minv_pattern_stride = x.minv_pattern_stride / 2;   // complex float -> float4 elements
    q.spectra = (float4 *)spectra;
    q.minv = (const float4 *)minv; q.tw1024 = (const float2 *)p.tw1024; q.twN = (const float2 *)p.twN;
    q.n_units = n_units; q.n_stations = n_stations; q.k_lo = p.k_lo; q.k_hi = p.k_hi; q.K = p.K;
    const int spec = spectra ? spec_mode : 0;
    const bool ef = efield != nullptr, i16 = x.input_i16 != 0, multi = x.pattern_id != nullptr;
    cudaError_t e;
    switch (w32_geom(p)) {
    case 0: e = launch_geom<10, 28, true>(q, s, ef, i16, multi, spec); break;
    case 1: e = launch_geom<6, 28, true>(q, s, ef, i16, multi, spec); break;
    default: e = launch_geom<0, 31, false>(q, s, ef, i16, multi, spec); break;
    }
    count_launches(1);
    return e;
}

} // namespace aera

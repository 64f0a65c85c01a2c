// Direction-hypothesis scan (BASELINE configs[2]) for N = 2048 fp32, built
// from the same warp-level pieces as unfold_w32.cu.
//
//   scan_fwd_w32_kernel : a2 ONCE per station. One warp per station: packed 1024-point forward
//       transform of the two polyphase halves, channel separation with the mirror bin, polyphase
//       fold; writes 2 V_c[k] on the band rows as float4 {V0.re, V0.im, V1.re, V1.im} to the
//       workspace, [station][band row][lane] (9.5 KB per station at configs[2], L2-resident).
//   scan_inv_w32_kernel : a4-a6 for every (direction, station) pair, peaks only. A CTA of 12 warps
//       works on tiles of 4 stations x 3 directions: warp w owns station 4 g + (w & 3) and keeps
//       that station's V in its tensor-memory columns for as long as the CTA stays in station group
//       g; the three directions' Minv (3 x 18 KB, contiguous in the workspace) arrive by ONE TMA
//       bulk copy per tile into a two-slot shared-memory ring, so the matrices of a direction are
//       read from L2 once per 4 stations and every warp's inner loop is: E = Minv V (registers),
//       two packed (theta, phi) pruned inverse transforms, env^2 running argmax, one 8-byte result.
//       No trace output: the kernel is pure FP32-pipe work.
//
// Tiles are ordered station-group-major and split into one contiguous range per CTA, so a CTA reloads V at
// most twice. Each CTA then streams its own part of the direction list: the 134 MB of per-direction matrices
// (configs[2]) do not fit the L2 next to each other, so they are read from DRAM once per station group
// (measured: 4.06 GB per launch, 0.9 TB/s = 14 % of the HBM peak, L2 hit rate 3 %). That costs nothing here
// (the kernel is bound by the FP32 pipe), and the L2-friendly orders tried in round 2 were SLOWER: direction
// blocks of 55 MB swept by all station groups (177 M pairs/s), chunks of 4..32 tiles dealt round-robin so that
// all CTAs work on the same few directions at the same time (178..188 M pairs/s) against 203 M pairs/s for this
// order -- 31 CTAs fetching the same 55 KB at the same moment queue up on the same L2 slices.
#include "w32_common.cuh"

namespace aera {
namespace {

constexpr int kScanStations = 4; // stations per tile; directions per tile: 3 (12 warps) when the tensor-memory columns allow, else 2

struct ScanParams {
    const float *traces;   // [S][2][2048]
    float4 *spectra;       // [S][band rows][32]
    const float4 *minv;    // [n_dirs] { A[K], B[K] } float4 (MINV_PACKED)
    float *amp;            // [n_dirs][S]
    int32_t *idx;
    const float2 *tw1024, *twN;
    long n_dirs;
    int n_stations;
    int k_lo, k_hi, K;
};

// ------------------------------------------------------------------------------------------------
// Kernel A: forward spectra, one warp per station.
template <int K2LO, int K2HI>
__global__ void __launch_bounds__(128, 1)
scan_fwd_w32_kernel(ScanParams p)
{
    using G = W32Geom<K2LO, K2HI>;
    extern __shared__ __align__(128) unsigned char smem[];
    float2 *T = reinterpret_cast<float2 *>(smem);
    float2 *TS = T + 1024;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    R *X = reinterpret_cast<R *>(smem + kTabBytes + (size_t)warp * G::kWarpBytes);
    R *QA = X, *QB = X + G::kPubRows * 32;
    for (int i = threadIdx.x; i < 1024; i += blockDim.x) {
        const int k1 = i >> 5, t = i & 31;
        T[i] = p.tw1024[(k1 * t) & 1023];
        TS[i] = p.twN[i];
    }
    __syncthreads();
    const int s = blockIdx.x * 4 + warp;
    if (s >= p.n_stations) return;
    const float *v = p.traces + (size_t)s * 4 * kM;
    R A[32], B[32];
    static_for<0, 32>([&](auto jc) {
        constexpr int j = decltype(jc)::value;
        A[brev5(j)] = ld_stream_b64(v + 2 * (lane + 32 * j));
        B[brev5(j)] = ld_stream_b64(v + 2 * kM + 2 * (lane + 32 * j));
    });
    fft1024(A, B, X, T, lane);
    static_for<G::kPubLo, G::kPubHi + 1>([&](auto rc) {
        constexpr int r = decltype(rc)::value;
        QA[(r - G::kPubLo) * 32 + lane] = A[r];
        QB[(r - G::kPubLo) * 32 + lane] = B[r];
    });
    __syncwarp();
    // same separation and polyphase fold as unfold_w32.cu's separate_solve, stopping at 2 V_c
    int own = (G::kLo - G::kPubLo) * 32 + lane;
    int par = (31 - G::kLo + (lane == 0 ? 1 : 0) - G::kPubLo) * 32 + ((32 - lane) & 31);
    int k = lane + 32 * G::kLo;
    float4 *out = p.spectra + (size_t)s * G::kBandRows * 32 + lane;
#pragma unroll 1
    for (int r = 0; r < G::kBandRows; ++r, own += 32, par -= 32, k += 32) {
        float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
        if (k >= p.k_lo && k <= p.k_hi) {
            const R ar = QA[own], ai = QB[own], pr = QA[par], pi = QB[par];
            const R f0r = L::add(ar, pr), f0i = L::sub(ai, pi);
            const R f1r = L::add(ai, pi), f1i = L::sub(pr, ar);
            float f0r0, f0r1, f0i0, f0i1, f1r0, f1r1, f1i0, f1i1;
            L::unpack(f0r, f0r0, f0r1); L::unpack(f0i, f0i0, f0i1);
            L::unpack(f1r, f1r0, f1r1); L::unpack(f1i, f1i0, f1i1);
            const float2 w = TS[k];
            o.x = fmaf(w.x, f0r1, f0r0); o.x = fmaf(-w.y, f0i1, o.x);
            o.y = fmaf(w.x, f0i1, f0i0); o.y = fmaf(w.y, f0r1, o.y);
            o.z = fmaf(w.x, f1r1, f1r0); o.z = fmaf(-w.y, f1i1, o.z);
            o.w = fmaf(w.x, f1i1, f1i0); o.w = fmaf(w.y, f1r1, o.w);
        }
        out[r * 32] = o;
    }
}

// ------------------------------------------------------------------------------------------------
// Kernel B: (direction, station) pairs.
template <int K2LO, int K2HI>
struct ScanGeom {
    using G = W32Geom<K2LO, K2HI>;
    static constexpr int kVCols = 4 * G::kBandRows;              // this station's 2 V_c, 4 columns per band row
    static constexpr int kCols = 2 * kVCols;                     // + the stash of E (read back for the odd samples)
    static constexpr int kDirs = 3 * kCols <= 512 ? 3 : 2;       // directions per tile: warps w, w+4(, w+8) share one TMEM lane quarter
    static constexpr int kWarps = kScanStations * kDirs;         // 12 (three warps per scheduler) or 8
    static constexpr int kColStride = 512 / kDirs;
    static_assert(kCols <= kColStride, "tensor-memory columns per warp");
    static constexpr bool kAnyBand = !G::kExact;                 // rows may lie wholly outside the band: clamp every Minv index
};

template <int K2LO, int K2HI>
__global__ void __launch_bounds__(ScanGeom<K2LO, K2HI>::kWarps * 32, 1)
scan_inv_w32_kernel(ScanParams p)
{
    using G = W32Geom<K2LO, K2HI>;
    using SG = ScanGeom<K2LO, K2HI>;
    constexpr int kWarps = SG::kWarps;
    constexpr int kScanDirs = SG::kDirs;
    extern __shared__ __align__(128) unsigned char smem[];
    float2 *T = reinterpret_cast<float2 *>(smem);
    float2 *TS = T + 1024;
    uint64_t *full = reinterpret_cast<uint64_t *>(smem + kTabBytes);
    int *done = reinterpret_cast<int *>(smem + kTabBytes + 16);
    uint32_t *tmem_base = reinterpret_cast<uint32_t *>(smem + kTabBytes + 32);
    const uint32_t minv_bytes = (uint32_t)p.K * 32u;
    const uint32_t slot_bytes = (kScanDirs * minv_bytes + 127u) & ~127u;
    unsigned char *mslot = smem + kTabBytes + kCtlBytes;
    const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
    const int lane = threadIdx.x & 31;
    const int wst = warp & 3, wdir = warp >> 2;
    R *X = reinterpret_cast<R *>(mslot + 2 * (size_t)slot_bytes + (size_t)warp * kXBytes);

    const long S = p.n_stations;
    const long n_groups = (S + kScanStations - 1) / kScanStations;
    const long n_trip = (p.n_dirs + kScanDirs - 1) / kScanDirs;
    const long n_tiles = n_groups * n_trip;
    const long i0 = n_tiles * (long)blockIdx.x / (long)gridDim.x;
    const long i1 = n_tiles * ((long)blockIdx.x + 1) / (long)gridDim.x;

    auto issue = [&](long i, int slot) { // one thread: Minv of tile i's directions -> ring slot
        const long t = i % n_trip;
        const long nd = p.n_dirs - kScanDirs * t < kScanDirs ? p.n_dirs - kScanDirs * t : kScanDirs;
        const uint32_t bytes = (uint32_t)nd * minv_bytes;
        mbar_expect_tx(&full[slot], bytes);
        tma_bulk_g2s(mslot + (size_t)slot * slot_bytes, p.minv + (size_t)(kScanDirs * t) * p.K * 2, bytes, &full[slot]);
    };

    if (warp == 0) tmem_alloc_all(tmem_base);
    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        done[0] = 0; done[1] = 0;
        for (int s = 0; s < 2 && i0 + s < i1; ++s) issue(i0 + s, s);
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
    const uint32_t tV = tmem_addr(tbase, warp, wdir * SG::kColStride);
    const uint32_t tstash = tV + SG::kVCols;

    long cur_g = -1;
#pragma unroll 1
    for (long i = i0; i < i1; ++i) {
        const int slot = (int)((i - i0) & 1);
        const uint32_t parity = (uint32_t)(((i - i0) >> 1) & 1);
        const long g = i / n_trip, t = i - g * n_trip;
        const long s = kScanStations * g + wst, d = kScanDirs * t + wdir;
        if (g != cur_g) { // new station group: this warp's station spectrum -> tensor memory
            cur_g = g;
            if (s < S) {
                const float4 *src = p.spectra + (size_t)s * G::kBandRows * 32 + lane;
#pragma unroll 1
                for (int r = 0; r < G::kBandRows; ++r) {
                    const float4 v = ld_nc_f4(src + r * 32);
                    tmem_st64(tV + 4 * r, L::pack(v.x, v.y).v);
                    tmem_st64(tV + 4 * r + 2, L::pack(v.z, v.w).v);
                }
                tmem_wait_st();
            }
        }
        mbar_wait(&full[slot], parity);
        if (s < S && d < p.n_dirs) {
            const float4 *MA = reinterpret_cast<const float4 *>(mslot + (size_t)slot * slot_bytes + (size_t)wdir * minv_bytes);
            const float4 *MB = MA + p.K;
            // ---- a4: E = Minv V on the band rows, straight into the even transform's input registers
            // (inverse roles: A = Im, B = Re) and into the tensor-memory stash for the odd transform
            R A[32], B[32];
            {
                unsigned long long vv[2 * G::kBandRows];
                static_for<0, G::kBandRows>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    vv[2 * r] = tmem_ld64(tV + 4 * r);
                    vv[2 * r + 1] = tmem_ld64(tV + 4 * r + 2);
                });
                tmem_wait_ld();
                static_for<0, G::kBandRows>([&](auto rc) {
                    constexpr int r = decltype(rc)::value;
                    tmem_ld_dep(vv[2 * r], vv[2 * r + 1]);
                });
                static_for<0, 32>([&](auto kc) {
                    constexpr int k2 = decltype(kc)::value;
                    if constexpr (k2 < G::kLo || k2 > G::kHi) { A[brev5(k2)] = L::zero(); B[brev5(k2)] = L::zero(); }
                    else {
                        constexpr int r = k2 - G::kLo;
                        int j = lane + 32 * k2 - p.k_lo; // edge rows: V is zero outside the band, keep the read in range
                        if (SG::kAnyBand || k2 == G::kLo) j = j < 0 ? 0 : j;
                        if (SG::kAnyBand || k2 == G::kHi) j = j > p.K - 1 ? p.K - 1 : j;
                        const float4 m0 = MA[j], m1 = MB[j];
                        const R Ma = L::pack(m0.x, m0.y), Mb = L::pack(m0.z, m0.w), Mc = L::pack(m1.x, m1.y), Md = L::pack(m1.z, m1.w);
                        float v0r, v0i, v1r, v1i;
                        R q0, q1; q0.v = vv[2 * r]; q1.v = vv[2 * r + 1];
                        L::unpack(q0, v0r, v0i); L::unpack(q1, v1r, v1i);
                        R er = L::mul(Ma, L::bc(v0r)); er = L::fma(Mb, L::bc(-v0i), er);
                        er = L::fma(Mc, L::bc(v1r), er); er = L::fma(Md, L::bc(-v1i), er);
                        R ei = L::mul(Ma, L::bc(v0i)); ei = L::fma(Mb, L::bc(v0r), ei);
                        ei = L::fma(Mc, L::bc(v1i), ei); ei = L::fma(Md, L::bc(v1r), ei);
                        B[brev5(k2)] = er; A[brev5(k2)] = ei;
                        tmem_st64(tstash + 4 * r, er.v);
                        tmem_st64(tstash + 4 * r + 2, ei.v);
                    }
                });
            }
            // ---- a5/a6: even samples, then odd samples, through ONE copy of the FFT code
            float best0 = -1.0f, best1 = -1.0f; int b0 = 0, b1 = 0;
            // bottom-tested loop with an opaque counter: ONE copy of the two-pass transform for the even (tpass = 1) and
            // the odd (tpass = 2) samples (a loop with the exit in the middle is rotated, which duplicates the transforms)
            int tpass = 1;
#pragma unroll 1
            do {
                // every transform of this kernel is an inverse one whose input is confined to the band rows: the first
                // pass runs the pruned 32-point transform (13 of its 16 first-stage butterflies are copies at configs[2])
                fft32_pruned<L, G::kLo, G::kHi>(A, B);
                pass_twiddle(A, B, T, lane);
                transpose_plane(A, X, lane);
                transpose_plane(B, X, lane);
                fft32<L>(A, B);
                asm volatile("" : "+r"(tpass));
                if (tpass == 1) {
                    emit_even<false>(B, A, 0u, best0, b0);
                    tmem_wait_st();
                    build_inverse_input<G, true>(B, A, TS, lane, tstash);
                } else
                    emit_odd<false>(B, A, lane, 0u, nullptr, best1, b1);
                ++tpass;
            } while (tpass <= 2);
            float best = best0; int bi = 2 * (lane + 32 * b0);
            {
                const int n1 = 2 * (lane + 32 * b1) + 1;
                if (best1 > best || (best1 == best && n1 < bi)) { best = best1; bi = n1; }
            }
            // env^2 >= 0: the float order is the order of the bit patterns, so two warp-wide integer reductions (REDUX)
            // give the maximum and the lowest index among the lanes that hold it
            {
                const unsigned bmax = __reduce_max_sync(0xffffffffu, __float_as_uint(best));
                bi = (int)__reduce_min_sync(0xffffffffu, __float_as_uint(best) == bmax ? (unsigned)bi : 0xffffffffu);
                best = __uint_as_float(bmax);
            }
            if (lane == 0) { p.amp[d * S + s] = sqrtf(best); p.idx[d * S + s] = bi; }
        }
        // ---- leave the tile: the last warp out refills the slot with the tile after next
        __syncwarp();
        if (lane == 0) {
            __threadfence_block();
            const int old = atomicAdd(&done[slot], 1);
            if (old == kWarps - 1) {
                done[slot] = 0;
                __threadfence_block();
                if (i + 2 < i1) {
                    fence_proxy_async_smem();
                    issue(i + 2, slot);
                }
            }
        }
    }
    tmem_fence_before_sync();
    __syncthreads();
    if (warp == 0) tmem_free_all(tbase);
}

} // namespace

bool scan_w32_supported(int dtype, const PlanDev &p)
{
    // rows 10..28 (30-80 MHz at fs = 180 MHz, configs[2]) have their own instantiation; <7, 27> and <0, 31> serve the other bands
    return dtype == AERA_F32 && p.N == 2 * kM && p.k_hi < kM && p.k_lo >= 1;
}

size_t scan_w32_spectra_bytes(int n_stations)
{
    return (size_t)n_stations * 32 * 32 * sizeof(float4);   // room for all 32 rows (any band)
}

template <int K2LO, int K2HI>
static cudaError_t launch_scan_inst(const ScanParams &q, cudaStream_t s)
{
    using G = W32Geom<K2LO, K2HI>;
    using SG = ScanGeom<K2LO, K2HI>;
    {
        ProfScope prof(KID_SCAN_FWD, s);
        const size_t smem = (size_t)kTabBytes + 4 * (size_t)G::kWarpBytes;
        auto kern = scan_fwd_w32_kernel<K2LO, K2HI>;
        AERA_ENSURE_DYN_SMEM(kern, smem);
        kern<<<(unsigned)((q.n_stations + 3) / 4), 128, smem, s>>>(q);
    }
    {
        ProfScope prof(KID_SCAN_INV, s);
        const size_t slot = ((size_t)SG::kDirs * q.K * 32 + 127) & ~(size_t)127;
        const size_t smem = (size_t)kTabBytes + kCtlBytes + 2 * slot + (size_t)SG::kWarps * kXBytes;
        auto kern = scan_inv_w32_kernel<K2LO, K2HI>;
        AERA_ENSURE_DYN_SMEM(kern, smem);
        const long n_tiles = (long)((q.n_stations + kScanStations - 1) / kScanStations) * ((q.n_dirs + SG::kDirs - 1) / SG::kDirs);
        const long grid = n_tiles < sm_count() ? n_tiles : sm_count();
        kern<<<(unsigned)grid, SG::kWarps * 32, smem, s>>>(q);
    }
    return cudaGetLastError();
}

cudaError_t launch_scan_w32(const PlanDev &p, int n_stations, const void *traces, long n_dirs, const void *minv,
                            void *amp, int32_t *idx, void *spectra, cudaStream_t s)
{
    if (n_dirs <= 0 || n_stations <= 0) return cudaSuccess;
    ScanParams q;
    q.traces = (const float *)traces; q.spectra = (float4 *)spectra; q.minv = (const float4 *)minv;
    q.amp = (float *)amp; q.idx = idx; q.tw1024 = (const float2 *)p.tw1024; q.twN = (const float2 *)p.twN;
    q.n_dirs = n_dirs; q.n_stations = n_stations; q.k_lo = p.k_lo; q.k_hi = p.k_hi; q.K = p.K;
    // <10, 28>: exactly configs[2]'s rows; <7, 27>: any band inside bins 224..895 (30-80 MHz at fs = 200-250 MHz), 21 rows:
    // still three directions per tile / twelve warps; <0, 31>: everything else (two directions per tile, eight warps)
    const int lo = p.k_lo >> 5, hi = p.k_hi >> 5;
    const cudaError_t e = (lo == 10 && hi == 28) ? launch_scan_inst<10, 28>(q, s)
                          : ((lo >= 7 && hi <= 27) ? launch_scan_inst<7, 27>(q, s) : launch_scan_inst<0, 31>(q, s));
    count_launches(2);
    return e;
}

} // namespace aera

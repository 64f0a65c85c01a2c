// C ABI of libaera_unfold.so (include/aera_unfold.h): argument validation, pattern handles,
// plan cache, workspace layout, kernel dispatch, and the host-buffer pipeline.
#include <atomic>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <utility>
#include <vector>

#include "aera_internal.h"

namespace aera {

static std::atomic<unsigned long long> g_launches{0};
static std::atomic<int> g_variant{0};
void count_launches(unsigned n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
int kernel_variant() { return g_variant.load(std::memory_order_relaxed); }

static thread_local char g_err[512] = "";
static thread_local const char *g_last_kernel = "";
void note_kernel(const char *name) { g_last_kernel = name; }

int sm_count()
{
    static std::atomic<int> cached[kMaxDevices];           // per device ordinal (zero = not asked yet)
    const int slot = device_slot();
    int n = slot >= 0 ? cached[slot].load(std::memory_order_relaxed) : 0;
    if (n > 0) return n;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) {
        (void)cudaGetLastError();
        n = 148; // B200
    }
    if (slot >= 0) cached[slot].store(n, std::memory_order_relaxed);
    return n;
}

// ---- per-kernel event timing -------------------------------------------------------------
struct ProfRec { int kid; cudaEvent_t e0, e1; };
static std::mutex g_prof_mu;
static std::atomic<int> g_prof_on{0};
static std::vector<ProfRec> g_prof_recs;
static std::vector<cudaEvent_t> g_prof_pool;
static thread_local cudaEvent_t g_prof_open = nullptr;

static cudaEvent_t prof_get_event()
{
    if (!g_prof_pool.empty()) { cudaEvent_t e = g_prof_pool.back(); g_prof_pool.pop_back(); return e; }
    cudaEvent_t e = nullptr;
    cudaEventCreate(&e);
    return e;
}
void prof_begin(int, cudaStream_t s)
{
    if (!g_prof_on.load(std::memory_order_relaxed)) return;
    std::lock_guard<std::mutex> lk(g_prof_mu);
    g_prof_open = prof_get_event();
    cudaEventRecord(g_prof_open, s);
}
void prof_end(int kid, cudaStream_t s)
{
    if (!g_prof_on.load(std::memory_order_relaxed) || !g_prof_open) return;
    std::lock_guard<std::mutex> lk(g_prof_mu);
    cudaEvent_t e1 = prof_get_event();
    cudaEventRecord(e1, s);
    g_prof_recs.push_back({kid, g_prof_open, e1});
    g_prof_open = nullptr;
}

static aera_status_t fail(aera_status_t st, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return st;
}
static aera_status_t cuda_fail(cudaError_t e, const char *what)
{
    return fail(AERA_ERR_CUDA, "%s: %s", what, cudaGetErrorString(e));
}

struct Plan {
    PlanDev dev{};
    double fs = 0;
    void *blob = nullptr; // one device allocation holding every table of the plan
};

struct HostPipe { // staging for aera_unfold_batch_host
    cudaStream_t st[3] = {nullptr, nullptr, nullptr};
    cudaEvent_t ev_in[2] = {nullptr, nullptr}, ev_k[2] = {nullptr, nullptr}, ev_out[2] = {nullptr, nullptr};
    void *d_in[2] = {nullptr, nullptr}, *d_out[2] = {nullptr, nullptr}, *d_amp[2] = {nullptr, nullptr};
    int32_t *d_idx[2] = {nullptr, nullptr};
    double *d_dirs[2] = {nullptr, nullptr};
    void *d_ws[2] = {nullptr, nullptr};
    size_t cap_units = 0, cap_in_bytes = 0, cap_out_bytes = 0, cap_ws = 0, cap_events = 0;
    bool ready = false;
};

} // namespace aera

using namespace aera;

struct aera_pattern {
    aera_pattern_desc_t desc{};
    void *d_table = nullptr;
    size_t table_bytes = 0;
    std::mutex mu;        // plans and filter weights
    std::mutex pipe_mu;   // the host pipeline's staging buffers and streams: one aera_unfold_batch_host at a time per handle
    std::map<std::pair<long long, double>, Plan *> plans;   // key: (n_samples | up-sampling factor << 32, fs)
    // optional per-bin pre-filter weights (aera_pattern_set_band_filter), device [K]; key: (n_samples, fs). The band does
    // not depend on the up-sampling factor, so every plan of (n_samples, fs) points its dev.bin_w at the same weights
    std::map<std::pair<long long, double>, double *> filters;
    HostPipe pipe;
};

namespace {

const size_t kAlign = 256;
size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }
size_t real_bytes(int dtype) { return dtype == AERA_F32 ? 4 : 8; }
size_t cplx_bytes(int dtype) { return 2 * real_bytes(dtype); }

bool is_whole(double x) { return x == std::floor(x) && std::fabs(x) < 9.0e15; }

int ilog2(int n)
{
    int l = 0;
    while ((1 << l) < n) ++l;
    return l;
}

aera_status_t check_n(int n_samples)
{
    if (n_samples < 64 || n_samples > 65536 || (n_samples & (n_samples - 1)) != 0)
        return fail(AERA_ERR_UNSUPPORTED_N, "n_samples=%d is not a power of two in [64, 65536]", n_samples);
    return AERA_OK;
}

// In-band bins: ceil(f0 N / fs) .. floor(f_hi N / fs), exact in integers for whole-Hz inputs.
aera_status_t compute_band(const aera_pattern_desc_t &d, int N, double fs, int *k_lo, int *k_hi)
{
    if (!(fs > 0) || !std::isfinite(fs)) return fail(AERA_ERR_INVALID_ARG, "fs_hz must be positive and finite");
    const double f_hi = d.freq0_hz + (d.n_freq - 1) * d.dfreq_hz;
    if (!(d.freq0_hz > 0) || !(f_hi < 0.5 * fs))
        return fail(AERA_ERR_BAND, "table band [%g, %g] Hz must lie strictly inside (0, fs/2 = %g)", d.freq0_hz, f_hi, 0.5 * fs);
    long long lo, hi;
    if (is_whole(fs) && is_whole(d.freq0_hz) && is_whole(d.dfreq_hz)) {
        const __int128 F = (long long)fs;
        const __int128 a = (__int128)(long long)d.freq0_hz * N;
        const __int128 b = ((__int128)(long long)d.freq0_hz + (__int128)(d.n_freq - 1) * (long long)d.dfreq_hz) * N;
        lo = (long long)((a + F - 1) / F);
        hi = (long long)(b / F);
    } else {
        lo = (long long)std::ceil((long double)d.freq0_hz * N / (long double)fs);
        hi = (long long)std::floor(((long double)d.freq0_hz + (long double)(d.n_freq - 1) * d.dfreq_hz) * N / (long double)fs);
    }
    if (lo < 1) lo = 1;
    if (hi > N / 2 - 1) hi = N / 2 - 1;
    if (hi < lo) return fail(AERA_ERR_BAND, "no DFT bin of N=%d, fs=%g falls inside the table band", N, fs);
    *k_lo = (int)lo;
    *k_hi = (int)hi;
    return AERA_OK;
}

template <typename T>
void fill_twiddles(cx<T> *dst, int count, int N)
{
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int m = 0; m < count; ++m) {
        long double a = two_pi * (long double)m / (long double)N;
        dst[m].re = (T)cosl(a);
        dst[m].im = (T)(-sinl(a));
    }
}

// Build (or fetch) the plan for (N, fs). May allocate and synchronise `s` on first use.
aera_status_t get_plan(aera_pattern *pat, int N, double fs, cudaStream_t s, Plan **out, int U = 1)
{
    std::lock_guard<std::mutex> lk(pat->mu);
    auto key = std::make_pair((long long)N | ((long long)U << 32), fs);
    auto it = pat->plans.find(key);
    if (it != pat->plans.end()) { *out = it->second; return AERA_OK; }

    int k_lo, k_hi;
    aera_status_t st = compute_band(pat->desc, N, fs, &k_lo, &k_hi);
    if (st != AERA_OK) return st;
    const int K = k_hi - k_lo + 1;
    const int dtype = pat->desc.dtype;
    const size_t cb = cplx_bytes(dtype);

    // blob layout: bin_if [K] | bin_tf [K] | tw [N/2] | tw1024 [1024] | twN [N] | twU [U N / 2] (U > 1 only)
    size_t off_if = 0;
    size_t off_tf = align_up(off_if + sizeof(int) * K);
    size_t off_tw = align_up(off_tf + sizeof(double) * K);
    size_t off_t1k = align_up(off_tw + cb * (N / 2));
    size_t off_twN = align_up(off_t1k + cb * 1024);
    size_t off_twU = align_up(off_twN + cb * N);
    size_t total = U > 1 ? align_up(off_twU + cb * ((size_t)U * N / 2)) : off_twU;
    std::vector<unsigned char> h(total, 0);
    int *bin_if = reinterpret_cast<int *>(h.data() + off_if);
    double *bin_tf = reinterpret_cast<double *>(h.data() + off_tf);
    for (int j = 0; j < K; ++j) {
        const double f = (double)(k_lo + j) * fs / (double)N;
        const double u = (f - pat->desc.freq0_hz) / pat->desc.dfreq_hz;
        int i = (int)std::floor(u);
        if (i > pat->desc.n_freq - 2) i = pat->desc.n_freq - 2;
        if (i < 0) i = 0;
        bin_if[j] = i;
        bin_tf[j] = u - (double)i;
    }
    if (dtype == AERA_F32) {
        fill_twiddles(reinterpret_cast<cx<float> *>(h.data() + off_tw), N / 2, N);
        fill_twiddles(reinterpret_cast<cx<float> *>(h.data() + off_t1k), 1024, 1024);
        fill_twiddles(reinterpret_cast<cx<float> *>(h.data() + off_twN), N, N);
        if (U > 1) fill_twiddles(reinterpret_cast<cx<float> *>(h.data() + off_twU), U * N / 2, U * N);
    } else {
        fill_twiddles(reinterpret_cast<cx<double> *>(h.data() + off_tw), N / 2, N);
        fill_twiddles(reinterpret_cast<cx<double> *>(h.data() + off_t1k), 1024, 1024);
        fill_twiddles(reinterpret_cast<cx<double> *>(h.data() + off_twN), N, N);
        if (U > 1) fill_twiddles(reinterpret_cast<cx<double> *>(h.data() + off_twU), U * N / 2, U * N);
    }
    Plan *pl = new (std::nothrow) Plan();
    if (!pl) return fail(AERA_ERR_ALLOC, "host allocation of a plan failed");
    cudaError_t e = cudaMalloc(&pl->blob, total);
    if (e != cudaSuccess) { delete pl; (void)cudaGetLastError(); return fail(AERA_ERR_ALLOC, "cudaMalloc(%zu) for a plan: %s", total, cudaGetErrorString(e)); }
    e = cudaMemcpyAsync(pl->blob, h.data(), total, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s); // h goes out of scope
    if (e != cudaSuccess) { cudaFree(pl->blob); delete pl; return cuda_fail(e, "plan upload"); }
    unsigned char *b = static_cast<unsigned char *>(pl->blob);
    pl->fs = fs;
    pl->dev.N = N; pl->dev.logN = ilog2(N);
    pl->dev.k_lo = k_lo; pl->dev.k_hi = k_hi; pl->dev.K = K;
    pl->dev.bin_if = reinterpret_cast<const int *>(b + off_if);
    pl->dev.bin_tf = reinterpret_cast<const double *>(b + off_tf);
    pl->dev.tw = b + off_tw;
    pl->dev.tw1024 = b + off_t1k;
    pl->dev.twN = b + off_twN;
    pl->dev.U = U; pl->dev.logM = ilog2(N * U);
    pl->dev.twU = U > 1 ? b + off_twU : b + off_tw;
    auto flt = pat->filters.find(std::make_pair((long long)N, fs));
    pl->dev.bin_w = flt != pat->filters.end() ? flt->second : nullptr;
    pat->plans[key] = pl;
    *out = pl;
    return AERA_OK;
}

TableGeom geom_of(const aera_pattern_desc_t &d)
{
    TableGeom g;
    g.n_z = d.n_zenith; g.n_a = d.n_azimuth; g.n_f = d.n_freq; g.periodic = d.azimuth_periodic ? 1 : 0;
    g.z0 = d.zenith0_deg; g.dz = d.dzenith_deg; g.a0 = d.azimuth0_deg; g.da = d.dazimuth_deg;
    return g;
}

struct WsLayout {
    size_t off_minv, off_scratch, off_spectra, off_loop_spectra, off_peaks, off_pid, total;
};

// Workspace: [Minv: n_dirs*K*4 complex] [generic transform buffers] [scan: spectra S*2*K complex]
WsLayout ws_layout(aera_op_t op, int dtype, int N, int k_lo, int K, long n_dirs, int n_stations, int n_patterns = 1, int upsample = 1)
{
    const int k_hi = k_lo + K - 1;
    PlanDev band{}; band.N = N; band.k_lo = k_lo; band.k_hi = k_hi; band.K = K;
    WsLayout w{};
    const size_t cb = cplx_bytes(dtype);
    size_t o = 0;
    size_t per_dir = (size_t)K * 4 + 8 * kMinvPad;                        // MINV_PACKED_PAD planes (covers MINV_Q4's + 32 too)
    const size_t q32 = (size_t)128 * ((k_hi >> 5) - (k_lo >> 5) + 1);     // MINV_Q32 planes
    if (q32 > per_dir) per_dir = q32;
    w.off_minv = o; o = align_up(o + (size_t)n_patterns * n_dirs * per_dir * cb);   // one slab of n_dirs matrices per table
    size_t scratch = generic_scratch_bytes(dtype, N, n_dirs * (long)n_stations, upsample);
    if (op != AERA_OP_SCAN && long_f32_supported(dtype, band) && long_f32_scratch_bytes(band) > scratch)
        scratch = long_f32_scratch_bytes(band);
    w.off_scratch = o; o = align_up(o + scratch);
    w.off_spectra = o;
    if (op == AERA_OP_SCAN) { // room for either scan path's station spectra
        size_t a = generic_scan_spectra_bytes(dtype, K, n_stations), b = scan_w32_spectra_bytes(n_stations);
        o = align_up(o + (a > b ? a : b));
    }
    w.off_loop_spectra = o;                                               // reconstruction loop: band spectra of every station
    if (op == AERA_OP_RECONSTRUCT && dtype == AERA_F32 && w32_supported(dtype, band))
        o = align_up(o + w32_spectra_bytes(band, n_dirs * (long)n_stations));
    w.off_peaks = o;                                                      // fold: the by-product peaks of the shared kernels
    if (op == AERA_OP_FOLD) o = align_up(o + (size_t)n_dirs * n_stations * 12);
    w.off_pid = o;                                                        // several tables: the range-checked copy of pattern_id
    if (n_patterns > 1) o = align_up(o + (size_t)n_stations * sizeof(int32_t));
    w.total = o > 0 ? o : kAlign;
    return w;
}

aera_status_t check_common(const aera_pattern_t *pattern, int dtype, int n_stations, int n_samples, double fs_hz)
{
    if (!pattern) return fail(AERA_ERR_INVALID_ARG, "pattern is NULL");
    if (dtype != AERA_F32 && dtype != AERA_F64) return fail(AERA_ERR_INVALID_ARG, "dtype=%d is neither AERA_F32 nor AERA_F64", dtype);
    if (dtype != pattern->desc.dtype) return fail(AERA_ERR_DTYPE_MISMATCH, "dtype=%d but the pattern was uploaded as dtype=%d", dtype, pattern->desc.dtype);
    if (n_stations <= 0) return fail(AERA_ERR_INVALID_ARG, "n_stations=%d must be positive", n_stations);
    aera_status_t st = check_n(n_samples);
    if (st != AERA_OK) return st;
    if (!(fs_hz > 0) || !std::isfinite(fs_hz)) return fail(AERA_ERR_INVALID_ARG, "fs_hz must be positive and finite");
    return AERA_OK;
}

bool misaligned(const void *p, size_t a) { return (reinterpret_cast<uintptr_t>(p) % a) != 0; }

} // namespace

extern "C" {

int aera_profile_enable(int on)
{
    std::lock_guard<std::mutex> lk(g_prof_mu);
    int prev = g_prof_on.exchange(on ? 1 : 0);
    if (on) {
        for (auto &r : g_prof_recs) { g_prof_pool.push_back(r.e0); g_prof_pool.push_back(r.e1); }
        g_prof_recs.clear();
    }
    return prev;
}

aera_status_t aera_profile_read(int kernel_id, double *total_ms, long *launches)
{
    if (!total_ms || !launches) return fail(AERA_ERR_INVALID_ARG, "total_ms and launches must be non-NULL");
    if (kernel_id < 0 || kernel_id >= KID_COUNT) return fail(AERA_ERR_INVALID_ARG, "kernel_id %d out of range", kernel_id);
    std::lock_guard<std::mutex> lk(g_prof_mu);
    double sum = 0; long n = 0;
    for (auto &r : g_prof_recs) {
        if (r.kid != kernel_id) continue;
        cudaError_t e = cudaEventSynchronize(r.e1);
        float ms = 0;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, r.e0, r.e1);
        if (e != cudaSuccess) return cuda_fail(e, "profile event read");
        sum += ms; ++n;
    }
    *total_ms = sum; *launches = n;
    return AERA_OK;
}

const char *aera_last_error(void) { return g_err; }
const char *aera_last_kernel(void) { return g_last_kernel; }
static const char *team_kernel_name(int dtype, int team_warps)
{
    if (team_warps == 4) return dtype == AERA_F64 ? "unfold_t4k_f64" : "unfold_t4k_f32";
    if (team_warps == 2) return dtype == AERA_F64 ? "unfold_t2k_f64" : "unfold_t2k_f32";
    if (team_warps == 8) return dtype == AERA_F64 ? "unfold_t8k_f64" : "unfold_t8k_f32";
    if (team_warps == 16) return "unfold_t16k_f32";
    return dtype == AERA_F64 ? "unfold_t1k_f64" : "unfold_t1k_f32";
}

aera_status_t aera_measure_alu_peak(int kind, int warps_per_sm, double *lane_fma_per_s, int *sm_count_out, int *sm_clock_khz)
{
    if (kind < 0 || kind > 2) return fail(AERA_ERR_INVALID_ARG, "kind=%d is not 0 (packed fp32), 1 (fp32) or 2 (fp64)", kind);
    if (warps_per_sm < 1 || warps_per_sm > 32) return fail(AERA_ERR_INVALID_ARG, "warps_per_sm=%d must be in 1..32", warps_per_sm);
    if (!lane_fma_per_s) return fail(AERA_ERR_INVALID_ARG, "lane_fma_per_s is NULL");
    int sms = 0, khz = 0;
    cudaError_t e = measure_alu_peak(kind, warps_per_sm, lane_fma_per_s, &sms, &khz);
    if (e != cudaSuccess) return cuda_fail(e, "ALU peak measurement");
    if (sm_count_out) *sm_count_out = sms;
    if (sm_clock_khz) *sm_clock_khz = khz;
    return AERA_OK;
}
const char *aera_version(void) { return "aera_unfold 0.1 (sm_100a)"; }
unsigned long long aera_launch_count(void) { return g_launches.load(); }
int aera_set_kernel_variant(int variant) { return g_variant.exchange(variant); }
int aera_set_long_trace_l2_persist(int megabytes) { return (int)set_long_persist_mb(megabytes); }

aera_status_t aera_pattern_upload(const aera_pattern_desc_t *desc, const void *H, int src_on_device,
                                  void *cuda_stream, aera_pattern_t **out)
{
    if (!desc || !H || !out) return fail(AERA_ERR_INVALID_ARG, "desc, H and out must be non-NULL");
    *out = nullptr;
    if (desc->dtype != AERA_F32 && desc->dtype != AERA_F64) return fail(AERA_ERR_INVALID_ARG, "desc->dtype=%d invalid", desc->dtype);
    if (desc->n_zenith < 2 || !(desc->dzenith_deg > 0)) return fail(AERA_ERR_INVALID_ARG, "zenith axis needs >= 2 nodes and a positive step");
    if (desc->n_azimuth < (desc->azimuth_periodic ? 3 : 2) || !(desc->dazimuth_deg > 0))
        return fail(AERA_ERR_INVALID_ARG, "azimuth axis needs >= %d nodes and a positive step", desc->azimuth_periodic ? 3 : 2);
    if (desc->n_freq < 2 || desc->n_freq > 512 || !(desc->dfreq_hz > 0) || !(desc->freq0_hz > 0))
        return fail(AERA_ERR_INVALID_ARG, "frequency axis needs 2..512 nodes, freq0 > 0 and a positive step");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    aera_pattern *p = new (std::nothrow) aera_pattern();
    if (!p) return fail(AERA_ERR_ALLOC, "host allocation of a pattern handle failed");
    p->desc = *desc;
    const size_t n = (size_t)4 * desc->n_zenith * desc->n_azimuth * desc->n_freq;
    p->table_bytes = n * cplx_bytes(desc->dtype);
    void *d_src = nullptr;
    cudaError_t e = cudaMalloc(&p->d_table, p->table_bytes);
    if (e != cudaSuccess) { delete p; (void)cudaGetLastError(); return fail(AERA_ERR_ALLOC, "cudaMalloc(%zu) for the table: %s", n, cudaGetErrorString(e)); }
    const void *src = H;
    if (!src_on_device) {
        e = cudaMalloc(&d_src, p->table_bytes);
        if (e != cudaSuccess) { cudaFree(p->d_table); delete p; (void)cudaGetLastError(); return fail(AERA_ERR_ALLOC, "cudaMalloc staging: %s", cudaGetErrorString(e)); }
        e = cudaMemcpyAsync(d_src, H, p->table_bytes, cudaMemcpyHostToDevice, s);
        if (e != cudaSuccess) { cudaFree(d_src); cudaFree(p->d_table); delete p; return cuda_fail(e, "table H2D copy"); }
        src = d_src;
    }
    e = launch_repack(desc->dtype, src, p->d_table, desc->n_zenith, desc->n_azimuth, desc->n_freq, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (d_src) cudaFree(d_src);
    if (e != cudaSuccess) { cudaFree(p->d_table); delete p; return cuda_fail(e, "table repack"); }
    *out = p;
    return AERA_OK;
}

aera_status_t aera_pattern_free(aera_pattern_t *p)
{
    if (!p) return AERA_OK;
    for (auto &kv : p->plans) { cudaFree(kv.second->blob); delete kv.second; }
    for (auto &kv : p->filters) cudaFree(kv.second);
    HostPipe &hp = p->pipe;
    for (int i = 0; i < 2; ++i) {
        cudaFree(hp.d_in[i]); cudaFree(hp.d_out[i]); cudaFree(hp.d_amp[i]); cudaFree(hp.d_idx[i]);
        cudaFree(hp.d_dirs[i]); cudaFree(hp.d_ws[i]);
        if (hp.ev_in[i]) cudaEventDestroy(hp.ev_in[i]);
        if (hp.ev_k[i]) cudaEventDestroy(hp.ev_k[i]);
        if (hp.ev_out[i]) cudaEventDestroy(hp.ev_out[i]);
    }
    for (int i = 0; i < 3; ++i) if (hp.st[i]) cudaStreamDestroy(hp.st[i]);
    cudaFree(p->d_table);
    delete p;
    return AERA_OK;
}

aera_status_t aera_band(const aera_pattern_t *pattern, int n_samples, double fs_hz, int *k_lo, int *k_hi)
{
    if (!pattern || !k_lo || !k_hi) return fail(AERA_ERR_INVALID_ARG, "pattern, k_lo and k_hi must be non-NULL");
    aera_status_t st = check_n(n_samples);
    if (st != AERA_OK) return st;
    return compute_band(pattern->desc, n_samples, fs_hz, k_lo, k_hi);
}

aera_status_t aera_pattern_set_band_filter(aera_pattern_t *pattern, int n_samples, double fs_hz, const double *weights,
                                           int n_weights, void *cuda_stream)
{
    if (!pattern) return fail(AERA_ERR_INVALID_ARG, "pattern is NULL");
    aera_status_t st = check_n(n_samples);
    if (st != AERA_OK) return st;
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    Plan *pl = nullptr;
    st = get_plan(pattern, n_samples, fs_hz, s, &pl);
    if (st != AERA_OK) return st;
    // a configuration call: no kernel of an earlier call on ANY stream (the host pipeline has its own) may still read the
    // old weights, and no other thread may build or fetch a plan of this pattern meanwhile
    std::lock_guard<std::mutex> lk(pattern->mu);
    cudaError_t e = cudaDeviceSynchronize();
    if (e != cudaSuccess) return cuda_fail(e, "device synchronise");
    const auto fkey = std::make_pair((long long)n_samples, fs_hz);
    // every plan of this (n_samples, fs_hz), whatever its up-sampling factor, uses the same weights
    auto point_plans_at = [&](const double *w) {
        for (auto &kv : pattern->plans)
            if ((kv.first.first & 0xffffffffLL) == (long long)n_samples && kv.first.second == fs_hz) kv.second->dev.bin_w = w;
    };
    auto cur = pattern->filters.find(fkey);
    if (!weights) {
        point_plans_at(nullptr);
        if (cur != pattern->filters.end()) { cudaFree(cur->second); pattern->filters.erase(cur); }
        return AERA_OK;
    }
    if (n_weights != pl->dev.K)
        return fail(AERA_ERR_INVALID_ARG, "n_weights=%d but the band of (n_samples=%d, fs=%g) has %d bins (aera_band)", n_weights, n_samples, fs_hz, pl->dev.K);
    for (int j = 0; j < n_weights; ++j)
        if (!std::isfinite(weights[j])) return fail(AERA_ERR_INVALID_ARG, "weights[%d] is not finite", j);
    double *d_w = cur != pattern->filters.end() ? cur->second : nullptr;
    if (!d_w) {
        e = cudaMalloc((void **)&d_w, sizeof(double) * pl->dev.K);
        if (e != cudaSuccess) { (void)cudaGetLastError(); return fail(AERA_ERR_ALLOC, "cudaMalloc of the filter weights: %s", cudaGetErrorString(e)); }
        pattern->filters[fkey] = d_w;
    }
    e = cudaMemcpyAsync(d_w, weights, sizeof(double) * pl->dev.K, cudaMemcpyHostToDevice, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return cuda_fail(e, "filter upload");
    point_plans_at(d_w);
    return AERA_OK;
}

size_t aera_workspace_bytes(aera_op_t op, const aera_pattern_t *pattern, int dtype, long n_events_or_dirs,
                            int n_stations, int n_samples, double fs_hz)
{
    if (op != AERA_OP_UNFOLD && op != AERA_OP_SCAN && op != AERA_OP_FOLD && op != AERA_OP_RECONSTRUCT) { fail(AERA_ERR_INVALID_ARG, "unknown op %d", (int)op); return 0; }
    if (check_common(pattern, dtype, n_stations, n_samples, fs_hz) != AERA_OK) return 0;
    if (n_events_or_dirs < 0) { fail(AERA_ERR_INVALID_ARG, "negative count"); return 0; }
    int k_lo, k_hi;
    if (compute_band(pattern->desc, n_samples, fs_hz, &k_lo, &k_hi) != AERA_OK) return 0;
    return ws_layout(op, dtype, n_samples, k_lo, k_hi - k_lo + 1, n_events_or_dirs, n_stations).total;
}

// Options of the variants that share unfold_impl
struct ImplExt {
    const aera_pattern_t *const *patterns = nullptr; // several resident tables (aera_unfold_batch_multi) ...
    int n_patterns = 1;
    const int32_t *pattern_id = nullptr;             // ... and the antenna type of each station (device)
    int input_i16 = 0;                               // traces are int16 ADC counts (aera_unfold_batch_i16)
    double g0 = 1.0, g1 = 1.0;                       // volts per count of the two channels
    int upsample = 1;                                // spectral up-sampling factor (aera_unfold_batch_upsampled)
};

// aera_unfold_batch (forward = 0) and aera_fold_batch (forward = 1: the same kernels with (1/N) H in place of
// (1/N) H^-1, peaks into the workspace), and the multi-table / int16 / up-sampled variants through `ext`
static aera_status_t unfold_impl(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                                 int n_samples, double fs_hz, const void *traces, const double *dirs,
                                 void *efield, void *peak_amp, int32_t *peak_idx,
                                 void *workspace, size_t workspace_bytes, void *cuda_stream, int forward, int spec_mode = 0,
                                 const ImplExt &ext = ImplExt())
{
    aera_status_t st = check_common(pattern, dtype, n_stations, n_samples, fs_hz);
    if (st != AERA_OK) return st;
    if (n_events < 0) return fail(AERA_ERR_INVALID_ARG, "n_events=%d is negative", n_events);
    if (n_events == 0) return AERA_OK;
    if (!traces || !dirs || (!forward && (!peak_amp || !peak_idx)) || (forward && !efield))
        return fail(AERA_ERR_INVALID_ARG, forward ? "efield, dirs and traces must be non-NULL" : "traces, dirs, peak_amp and peak_idx must be non-NULL");
    if (misaligned(traces, 16) || (efield && misaligned(efield, 16))) return fail(AERA_ERR_INVALID_ARG, "traces and efield must be 16-byte aligned");
    if (misaligned(dirs, 8) || (!forward && (misaligned(peak_amp, real_bytes(dtype)) || misaligned(peak_idx, 4))))
        return fail(AERA_ERR_INVALID_ARG, "dirs / peak_amp / peak_idx are not aligned to their element size");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    Plan *pl = nullptr;
    st = get_plan(const_cast<aera_pattern *>(pattern), n_samples, fs_hz, s, &pl, ext.upsample);
    if (st != AERA_OK) return st;
    const WsLayout w = ws_layout(forward ? AERA_OP_FOLD : (spec_mode ? AERA_OP_RECONSTRUCT : AERA_OP_UNFOLD), dtype, n_samples,
                                 pl->dev.k_lo, pl->dev.K, n_events, n_stations, ext.n_patterns, ext.upsample);
    if (!workspace || misaligned(workspace, kAlign) || workspace_bytes < w.total)
        return fail(AERA_ERR_WORKSPACE, "workspace must be non-NULL, 256-byte aligned and >= %zu bytes (got %zu)", w.total, workspace_bytes);
    unsigned char *ws = static_cast<unsigned char *>(workspace);
    if (forward) { // the kernels' envelope peaks are a by-product here: they go to the workspace
        peak_amp = ws + w.off_peaks;
        peak_idx = reinterpret_cast<int32_t *>(ws + w.off_peaks + (size_t)n_events * n_stations * 8);
    }

    // up-sampling runs on the generic kernels (the specialised ones transform on the input grid only)
    const bool fast = kernel_variant() == 0 && ext.upsample == 1;
    const bool warp_path = fast && w32_supported(dtype, pl->dev);
    const bool team_path = fast && t4k_supported(dtype, pl->dev);   // (int16 input: fp32 only, which aera_unfold_batch_i16 guarantees)
    const bool long_path = fast && !ext.input_i16 && long_f32_supported(dtype, pl->dev);
    const int team_warps = team_path ? t4k_team_warps(dtype, pl->dev) : 0;
    const int layout = warp_path ? MINV_PACKED_PAD
                                 : (team_path ? (team_warps == 4 ? MINV_Q4 : (team_warps == 2 ? MINV_Q2 : (team_warps == 8 ? MINV_Q8 : (team_warps == 16 ? MINV_Q16 : MINV_Q1)))) : (long_path ? MINV_Q32 : MINV_ROWS));
    // complex elements of one event's matrices in this layout; the tables' slabs follow one another
    const size_t per_event = team_path ? minv_qt_stride(team_warps, pl->dev.k_lo, pl->dev.k_hi)
                             : (layout == MINV_Q32 ? (size_t)128 * ((pl->dev.k_hi >> 5) - (pl->dev.k_lo >> 5) + 1)
                                                   : (layout == MINV_PACKED_PAD ? (size_t)(pl->dev.K + 2 * kMinvPad) * 4 : (size_t)pl->dev.K * 4));
    UnfoldExt x;
    x.pattern_id = ext.pattern_id;
    if (ext.pattern_id && ext.n_patterns > 1) {   // the kernels index the matrix slabs with it: hand them a copy forced into range
        int32_t *pid = reinterpret_cast<int32_t *>(ws + w.off_pid);
        cudaError_t ce = launch_clamp_pattern_id(ext.pattern_id, pid, n_stations, ext.n_patterns, s);
        if (ce != cudaSuccess) return cuda_fail(ce, "pattern_id range check launch");
        x.pattern_id = pid;
    } else if (ext.n_patterns == 1) {
        x.pattern_id = nullptr;                    // one table: whatever the ids say, every station uses it
    }
    x.minv_pattern_stride = (size_t)n_events * per_event;
    x.input_i16 = ext.input_i16;
    // the warp, team and long kernels form 2 V_c, so their matrix carries 1/N instead of 2/N
    const double scale = ((warp_path || team_path || long_path) ? 1.0 : 2.0) / (double)n_samples;
    cudaError_t e = cudaSuccess;
    for (int t = 0; t < ext.n_patterns && e == cudaSuccess; ++t) {
        const aera_pattern_t *pt = ext.patterns ? ext.patterns[t] : pattern;
        e = launch_minv(dtype, pt->d_table, geom_of(pt->desc), pl->dev, dirs, n_events,
                        ws + w.off_minv + (size_t)t * x.minv_pattern_stride * cplx_bytes(dtype), layout, scale, s, forward, ext.g0, ext.g1);
    }
    if (e != cudaSuccess) return cuda_fail(e, "minv kernel launch");
    note_kernel(warp_path ? "unfold_w32" : (team_path ? team_kernel_name(dtype, team_warps) : (long_path ? "unfold_long_f32" : "generic")));
    if (warp_path)
        e = launch_unfold_w32(pl->dev, n_events, n_stations, traces, efield, peak_amp, peak_idx, ws + w.off_minv, s,
                              spec_mode ? ws + w.off_loop_spectra : nullptr, spec_mode, x);
    else if (team_path)
        e = launch_unfold_t4k(dtype, pl->dev, n_events, n_stations, traces, efield, peak_amp, peak_idx, ws + w.off_minv, s, x);
    else if (long_path)
        e = launch_unfold_long_f32(pl->dev, n_events, n_stations, traces, efield, peak_amp, peak_idx, ws + w.off_minv,
                                   ws + w.off_scratch, s, x);
    else
        e = launch_unfold_generic(dtype, pl->dev, n_events, n_stations, traces, efield, peak_amp, peak_idx,
                                  ws + w.off_minv, ws + w.off_scratch, s, x);
    if (e != cudaSuccess) return cuda_fail(e, "unfold kernel launch");
    return AERA_OK;
}

aera_status_t aera_unfold_batch(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                                int n_samples, double fs_hz, const void *traces, const double *dirs,
                                void *efield, void *peak_amp, int32_t *peak_idx,
                                void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    return unfold_impl(pattern, dtype, n_events, n_stations, n_samples, fs_hz, traces, dirs, efield, peak_amp, peak_idx,
                       workspace, workspace_bytes, cuda_stream, 0);
}

aera_status_t aera_fold_batch(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                              int n_samples, double fs_hz, const void *efield, const double *dirs,
                              void *traces, void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    // the kernels read their "traces" argument and write their "efield" argument: swapped roles here
    return unfold_impl(pattern, dtype, n_events, n_stations, n_samples, fs_hz, efield, dirs, traces, nullptr, nullptr,
                       workspace, workspace_bytes, cuda_stream, 1);
}

// ---- several tables, one antenna type per station
static aera_status_t check_patterns(const aera_pattern_t *const *patterns, int n_patterns)
{
    if (!patterns || n_patterns < 1 || n_patterns > 64) return fail(AERA_ERR_INVALID_ARG, "patterns must be non-NULL and 1 <= n_patterns <= 64");
    for (int t = 0; t < n_patterns; ++t) {
        if (!patterns[t]) return fail(AERA_ERR_INVALID_ARG, "patterns[%d] is NULL", t);
        const aera_pattern_desc_t &a = patterns[0]->desc, &b = patterns[t]->desc;
        if (a.dtype != b.dtype) return fail(AERA_ERR_DTYPE_MISMATCH, "patterns[%d] has another dtype than patterns[0]", t);
        if (a.n_freq != b.n_freq || a.freq0_hz != b.freq0_hz || a.dfreq_hz != b.dfreq_hz)
            return fail(AERA_ERR_INVALID_ARG, "patterns[%d] has another frequency axis than patterns[0] (the in-band bins must agree)", t);
    }
    return AERA_OK;
}

size_t aera_workspace_bytes_ex(aera_op_t op, const aera_pattern_t *pattern, int dtype, long n_events_or_dirs,
                               int n_stations, int n_samples, double fs_hz, int n_patterns, int upsample)
{
    if (op != AERA_OP_UNFOLD && op != AERA_OP_SCAN && op != AERA_OP_FOLD && op != AERA_OP_RECONSTRUCT) { fail(AERA_ERR_INVALID_ARG, "unknown op %d", (int)op); return 0; }
    if (check_common(pattern, dtype, n_stations, n_samples, fs_hz) != AERA_OK) return 0;
    if (n_events_or_dirs < 0 || n_patterns < 1 || n_patterns > 64) { fail(AERA_ERR_INVALID_ARG, "negative count or n_patterns outside 1..64"); return 0; }
    if (upsample < 1 || (upsample & (upsample - 1)) != 0 || (long)upsample * n_samples > 65536) { fail(AERA_ERR_INVALID_ARG, "upsample=%d must be a power of two with upsample * n_samples <= 65536", upsample); return 0; }
    int k_lo, k_hi;
    if (compute_band(pattern->desc, n_samples, fs_hz, &k_lo, &k_hi) != AERA_OK) return 0;
    return ws_layout(op, dtype, n_samples, k_lo, k_hi - k_lo + 1, n_events_or_dirs, n_stations, n_patterns, upsample).total;
}

aera_status_t aera_unfold_batch_multi(const aera_pattern_t *const *patterns, int n_patterns, const int32_t *pattern_id,
                                      int dtype, int n_events, int n_stations, int n_samples, double fs_hz,
                                      const void *traces, const double *dirs, void *efield, void *peak_amp, int32_t *peak_idx,
                                      void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    aera_status_t st = check_patterns(patterns, n_patterns);
    if (st != AERA_OK) return st;
    if (!pattern_id || misaligned(pattern_id, 4)) return fail(AERA_ERR_INVALID_ARG, "pattern_id must be a non-NULL, 4-byte aligned device pointer");
    ImplExt ext;
    ext.patterns = patterns; ext.n_patterns = n_patterns; ext.pattern_id = pattern_id;
    return unfold_impl(patterns[0], dtype, n_events, n_stations, n_samples, fs_hz, traces, dirs, efield, peak_amp, peak_idx,
                       workspace, workspace_bytes, cuda_stream, 0, 0, ext);
}

// ---- int16 ADC-count input, spectral up-sampling
aera_status_t aera_unfold_batch_i16(const aera_pattern_t *pattern, int n_events, int n_stations, int n_samples, double fs_hz,
                                    const int16_t *traces, const double *counts_to_volts, const double *dirs,
                                    float *efield, float *peak_amp, int32_t *peak_idx,
                                    void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (!counts_to_volts || !std::isfinite(counts_to_volts[0]) || !std::isfinite(counts_to_volts[1]))
        return fail(AERA_ERR_INVALID_ARG, "counts_to_volts must point to two finite factors (host memory)");
    ImplExt ext;
    ext.input_i16 = 1; ext.g0 = counts_to_volts[0]; ext.g1 = counts_to_volts[1];
    return unfold_impl(pattern, AERA_F32, n_events, n_stations, n_samples, fs_hz, traces, dirs, efield, peak_amp, peak_idx,
                       workspace, workspace_bytes, cuda_stream, 0, 0, ext);
}

aera_status_t aera_unfold_batch_upsampled(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations, int n_samples,
                                          double fs_hz, int upsample, const void *traces, const double *dirs,
                                          void *efield, void *peak_amp, int32_t *peak_idx,
                                          void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    if (upsample < 1 || (upsample & (upsample - 1)) != 0 || (long)upsample * n_samples > 65536)
        return fail(AERA_ERR_INVALID_ARG, "upsample=%d must be a power of two with upsample * n_samples <= 65536", upsample);
    ImplExt ext;
    ext.upsample = upsample;
    return unfold_impl(pattern, dtype, n_events, n_stations, n_samples, fs_hz, traces, dirs, efield, peak_amp, peak_idx,
                       workspace, workspace_bytes, cuda_stream, 0, 0, ext);
}

aera_status_t aera_scan_directions(const aera_pattern_t *pattern, int dtype, int n_stations, int n_samples,
                                   double fs_hz, const void *traces, long n_dirs, const double *dirs,
                                   void *peak_amp, int32_t *peak_idx,
                                   void *workspace, size_t workspace_bytes, void *cuda_stream)
{
    aera_status_t st = check_common(pattern, dtype, n_stations, n_samples, fs_hz);
    if (st != AERA_OK) return st;
    if (n_dirs < 0) return fail(AERA_ERR_INVALID_ARG, "n_dirs=%ld is negative", n_dirs);
    if (n_dirs == 0) return AERA_OK;
    if (n_dirs > 0x7fffffffL / 4) return fail(AERA_ERR_INVALID_ARG, "n_dirs=%ld too large", n_dirs);
    if (!traces || !dirs || !peak_amp || !peak_idx) return fail(AERA_ERR_INVALID_ARG, "traces, dirs, peak_amp and peak_idx must be non-NULL");
    if (misaligned(traces, 16)) return fail(AERA_ERR_INVALID_ARG, "traces must be 16-byte aligned");
    if (misaligned(dirs, 8) || misaligned(peak_amp, real_bytes(dtype)) || misaligned(peak_idx, 4))
        return fail(AERA_ERR_INVALID_ARG, "dirs / peak_amp / peak_idx are not aligned to their element size");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    Plan *pl = nullptr;
    st = get_plan(const_cast<aera_pattern *>(pattern), n_samples, fs_hz, s, &pl);
    if (st != AERA_OK) return st;
    const WsLayout w = ws_layout(AERA_OP_SCAN, dtype, n_samples, pl->dev.k_lo, pl->dev.K, n_dirs, n_stations);
    if (!workspace || misaligned(workspace, kAlign) || workspace_bytes < w.total)
        return fail(AERA_ERR_WORKSPACE, "workspace must be non-NULL, 256-byte aligned and >= %zu bytes (got %zu)", w.total, workspace_bytes);
    unsigned char *ws = static_cast<unsigned char *>(workspace);

    const bool warp_path = kernel_variant() == 0 && scan_w32_supported(dtype, pl->dev);
    cudaError_t e = launch_minv(dtype, pattern->d_table, geom_of(pattern->desc), pl->dev, dirs, n_dirs, ws + w.off_minv,
                                warp_path ? MINV_PACKED : MINV_ROWS, (warp_path ? 1.0 : 2.0) / (double)n_samples, s);
    if (e != cudaSuccess) return cuda_fail(e, "minv kernel launch");
    note_kernel(warp_path ? "scan_w32" : "generic");
    if (warp_path)
        e = launch_scan_w32(pl->dev, n_stations, traces, n_dirs, ws + w.off_minv, peak_amp, peak_idx, ws + w.off_spectra, s);
    else
        e = launch_scan_generic(dtype, pl->dev, n_stations, traces, n_dirs, ws + w.off_minv, peak_amp, peak_idx,
                                ws + w.off_spectra, ws + w.off_scratch, s);
    if (e != cudaSuccess) return cuda_fail(e, "scan kernel launch");
    return AERA_OK;
}

aera_status_t aera_reconstruct_batch(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                                     int n_samples, double fs_hz, const void *traces, const double *positions,
                                     int n_iter, double *dirs_hist, void *efield, void *amp_hist, int32_t *idx_hist,
                                     int32_t *idx0, void *w0, void *workspace, size_t workspace_bytes,
                                     void *cuda_stream)
{
    aera_status_t st = check_common(pattern, dtype, n_stations, n_samples, fs_hz);
    if (st != AERA_OK) return st;
    if (n_events < 0) return fail(AERA_ERR_INVALID_ARG, "n_events=%d is negative", n_events);
    if (n_iter < 1) return fail(AERA_ERR_INVALID_ARG, "n_iter=%d must be at least 1", n_iter);
    if (n_events == 0) return AERA_OK;
    if (!traces || !positions || !dirs_hist || !amp_hist || !idx_hist || !idx0 || !w0)
        return fail(AERA_ERR_INVALID_ARG, "traces, positions, dirs_hist, amp_hist, idx_hist, idx0 and w0 must be non-NULL");
    if (misaligned(traces, 16) || misaligned(positions, 8) || misaligned(dirs_hist, 8))
        return fail(AERA_ERR_INVALID_ARG, "traces must be 16-byte aligned, positions and dirs_hist 8-byte aligned");
    cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
    const size_t rb = real_bytes(dtype);
    const size_t units = (size_t)n_events * n_stations;
    cudaError_t e = launch_timing(dtype, traces, (long)units, n_samples, idx0, w0, s);
    if (e != cudaSuccess) return cuda_fail(e, "timing kernel launch");
    // spectrum reuse (fp32 warp kernel only): needs the larger AERA_OP_RECONSTRUCT workspace
    bool reuse = false;
    if (n_iter > 1 && kernel_variant() == 0 && dtype == AERA_F32) {
        int k_lo, k_hi;
        if (compute_band(pattern->desc, n_samples, fs_hz, &k_lo, &k_hi) == AERA_OK) {
            PlanDev band{}; band.N = n_samples; band.k_lo = k_lo; band.k_hi = k_hi; band.K = k_hi - k_lo + 1;
            reuse = w32_supported(dtype, band) && w32_spectra_bytes(band, (long)units) > 0 &&
                    workspace_bytes >= ws_layout(AERA_OP_RECONSTRUCT, dtype, n_samples, k_lo, band.K, n_events, n_stations).total;
        }
    }
    const int32_t *t_idx = idx0;
    const void *t_w = w0;
    int square = 0;
    for (int it = 0; it < n_iter; ++it) {
        double *dirs = dirs_hist + (size_t)it * n_events * 2;
        e = launch_planefit(dtype, positions, t_idx, t_w, square, n_events, n_stations, fs_hz, dirs, s);
        if (e != cudaSuccess) return cuda_fail(e, "plane-wave fit kernel launch");
        void *amp = static_cast<unsigned char *>(amp_hist) + (size_t)it * units * rb;
        int32_t *idx = idx_hist + (size_t)it * units;
        st = unfold_impl(pattern, dtype, n_events, n_stations, n_samples, fs_hz, traces, dirs,
                         it == n_iter - 1 ? efield : nullptr, amp, idx, workspace, workspace_bytes, cuda_stream, 0,
                         reuse ? (it == 0 ? 1 : 2) : 0);
        if (st != AERA_OK) return st;
        t_idx = idx; t_w = amp; square = 1;
    }
    return AERA_OK;
}

aera_status_t aera_reconstruct_convergence(const double *dirs_hist, int n_iter, int n_events, double tol_deg, int32_t *conv_iter, void *cuda_stream)
{
    if (!dirs_hist || !conv_iter) return fail(AERA_ERR_INVALID_ARG, "dirs_hist and conv_iter must be non-NULL");
    if (n_iter < 1 || n_events < 0 || !(tol_deg > 0)) return fail(AERA_ERR_INVALID_ARG, "n_iter >= 1, n_events >= 0 and tol_deg > 0 are required");
    cudaError_t e = launch_convergence(dirs_hist, n_iter, n_events, tol_deg, conv_iter, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(e, "convergence kernel launch");
    return AERA_OK;
}

// aera_unfold_batch_host (in_i16 = 0) and aera_unfold_batch_host_i16 (in_i16 = 1: int16 ADC counts in, fp32 out)
static aera_status_t host_impl(aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                               int n_samples, double fs_hz, const void *traces_host, int in_i16, const double *counts_to_volts,
                               const double *dirs_host, void *efield_host, void *peak_amp_host,
                               int32_t *peak_idx_host)
{
    aera_status_t st = check_common(pattern, dtype, n_stations, n_samples, fs_hz);
    if (st != AERA_OK) return st;
    if (n_events < 0) return fail(AERA_ERR_INVALID_ARG, "n_events=%d is negative", n_events);
    if (n_events == 0) return AERA_OK;
    if (!traces_host || !dirs_host || !peak_amp_host || !peak_idx_host)
        return fail(AERA_ERR_INVALID_ARG, "traces, dirs, peak_amp and peak_idx must be non-NULL");

    const size_t rb = real_bytes(dtype);
    const size_t unit_bytes = (size_t)2 * n_samples * rb;
    const size_t event_bytes = unit_bytes * n_stations;                                   // one event of E-field output
    const size_t event_in_bytes = in_i16 ? (size_t)2 * n_samples * sizeof(int16_t) * n_stations : event_bytes;
    // chunk: ~64 MB of traces per stage (AERA_HOST_CHUNK_MB overrides, tuning only), at least one event
    static const size_t chunk_mb = [] { const char *e = getenv("AERA_HOST_CHUNK_MB"); const int v = e ? atoi(e) : 64; return (size_t)(v < 1 ? 1 : (v > 1024 ? 1024 : v)); }();
    long chunk_events = (long)((chunk_mb << 20) / event_bytes);
    if (chunk_events < 1) chunk_events = 1;
    if (chunk_events > n_events) chunk_events = n_events;

    std::lock_guard<std::mutex> pipe_lock(pattern->pipe_mu);
    HostPipe &hp = pattern->pipe;
    cudaError_t e;
    // every error exit below first drains the three streams: no copy into the caller's buffers may be in flight on return
    auto drained = [&](aera_status_t st_) { for (int i = 0; i < 3; ++i) if (hp.st[i]) cudaStreamSynchronize(hp.st[i]); return st_; };
    if (!hp.ready) {
        for (int i = 0; i < 3; ++i) { e = cudaStreamCreateWithFlags(&hp.st[i], cudaStreamNonBlocking); if (e != cudaSuccess) return cuda_fail(e, "stream create"); }
        for (int i = 0; i < 2; ++i) {
            if ((e = cudaEventCreateWithFlags(&hp.ev_in[i], cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e, "event create");
            if ((e = cudaEventCreateWithFlags(&hp.ev_k[i], cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e, "event create");
            if ((e = cudaEventCreateWithFlags(&hp.ev_out[i], cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e, "event create");
        }
        hp.ready = true;
    }
    Plan *pl = nullptr;
    st = get_plan(pattern, n_samples, fs_hz, hp.st[1], &pl);
    if (st != AERA_OK) return st;
    const size_t need_in = (size_t)chunk_events * event_in_bytes;
    const size_t need_out = efield_host ? (size_t)chunk_events * event_bytes : 0;          // peaks only: no E-field staging at all
    const size_t need_units = (size_t)chunk_events * n_stations;
    const size_t need_ws = ws_layout(AERA_OP_UNFOLD, dtype, n_samples, pl->dev.k_lo, pl->dev.K, chunk_events, n_stations).total;
    if (need_in > hp.cap_in_bytes || need_out > hp.cap_out_bytes || need_units > hp.cap_units || need_ws > hp.cap_ws || (size_t)chunk_events > hp.cap_events) {
        const size_t new_in = need_in > hp.cap_in_bytes ? need_in : hp.cap_in_bytes, new_out = need_out > hp.cap_out_bytes ? need_out : hp.cap_out_bytes;
        cudaDeviceSynchronize();
        for (int i = 0; i < 2; ++i) {
            cudaFree(hp.d_in[i]); cudaFree(hp.d_out[i]); cudaFree(hp.d_amp[i]); cudaFree(hp.d_idx[i]); cudaFree(hp.d_dirs[i]); cudaFree(hp.d_ws[i]);
            hp.d_in[i] = hp.d_out[i] = hp.d_amp[i] = hp.d_ws[i] = nullptr; hp.d_idx[i] = nullptr; hp.d_dirs[i] = nullptr;
            bool ok = cudaMalloc(&hp.d_in[i], new_in) == cudaSuccess && (new_out == 0 || cudaMalloc(&hp.d_out[i], new_out) == cudaSuccess) &&
                      cudaMalloc(&hp.d_amp[i], need_units * 8) == cudaSuccess && cudaMalloc((void **)&hp.d_idx[i], need_units * 4) == cudaSuccess &&
                      cudaMalloc((void **)&hp.d_dirs[i], (size_t)chunk_events * 16) == cudaSuccess && cudaMalloc(&hp.d_ws[i], need_ws) == cudaSuccess;
            if (!ok) { (void)cudaGetLastError(); hp.cap_in_bytes = hp.cap_out_bytes = hp.cap_units = hp.cap_ws = hp.cap_events = 0; return fail(AERA_ERR_ALLOC, "cudaMalloc of host-pipeline staging buffers failed"); }
        }
        hp.cap_in_bytes = new_in; hp.cap_out_bytes = new_out; hp.cap_units = need_units; hp.cap_ws = need_ws; hp.cap_events = (size_t)chunk_events;
    }

    const unsigned char *tin = static_cast<const unsigned char *>(traces_host);
    unsigned char *eout = static_cast<unsigned char *>(efield_host);
    unsigned char *aout = static_cast<unsigned char *>(peak_amp_host);
    long done = 0; int it = 0;
    while (done < n_events) {
        const int b = it & 1;
        const long ne = (n_events - done < chunk_events) ? (n_events - done) : chunk_events;
        const size_t units = (size_t)ne * n_stations;
        // stage b's input buffer is free once the kernel that read it (2 iterations ago) finished;
        // its output buffers are free once their D2H copy finished.
        if (it >= 2) {
            if ((e = cudaStreamWaitEvent(hp.st[0], hp.ev_k[b], 0)) != cudaSuccess) return drained(cuda_fail(e, "stream wait"));
            if ((e = cudaStreamWaitEvent(hp.st[1], hp.ev_out[b], 0)) != cudaSuccess) return drained(cuda_fail(e, "stream wait"));
        }
        if ((e = cudaMemcpyAsync(hp.d_in[b], tin + (size_t)done * event_in_bytes, (size_t)ne * event_in_bytes, cudaMemcpyHostToDevice, hp.st[0])) != cudaSuccess) return drained(cuda_fail(e, "H2D traces"));
        if ((e = cudaMemcpyAsync(hp.d_dirs[b], dirs_host + 2 * done, (size_t)ne * 16, cudaMemcpyHostToDevice, hp.st[0])) != cudaSuccess) return drained(cuda_fail(e, "H2D dirs"));
        cudaEventRecord(hp.ev_in[b], hp.st[0]);
        cudaStreamWaitEvent(hp.st[1], hp.ev_in[b], 0);
        if (in_i16)
            st = aera_unfold_batch_i16(pattern, (int)ne, n_stations, n_samples, fs_hz, static_cast<const int16_t *>(hp.d_in[b]), counts_to_volts,
                                       hp.d_dirs[b], efield_host ? static_cast<float *>(hp.d_out[b]) : nullptr, static_cast<float *>(hp.d_amp[b]),
                                       hp.d_idx[b], hp.d_ws[b], hp.cap_ws, hp.st[1]);
        else
            st = aera_unfold_batch(pattern, dtype, (int)ne, n_stations, n_samples, fs_hz, hp.d_in[b], hp.d_dirs[b],
                                   efield_host ? hp.d_out[b] : nullptr, hp.d_amp[b], hp.d_idx[b], hp.d_ws[b], hp.cap_ws, hp.st[1]);
        if (st != AERA_OK) return drained(st);
        cudaEventRecord(hp.ev_k[b], hp.st[1]);
        cudaStreamWaitEvent(hp.st[2], hp.ev_k[b], 0);
        if (efield_host)
            if ((e = cudaMemcpyAsync(eout + (size_t)done * event_bytes, hp.d_out[b], (size_t)ne * event_bytes, cudaMemcpyDeviceToHost, hp.st[2])) != cudaSuccess) return drained(cuda_fail(e, "D2H efield"));
        if ((e = cudaMemcpyAsync(aout + (size_t)done * n_stations * rb, hp.d_amp[b], units * rb, cudaMemcpyDeviceToHost, hp.st[2])) != cudaSuccess) return drained(cuda_fail(e, "D2H amp"));
        if ((e = cudaMemcpyAsync(peak_idx_host + (size_t)done * n_stations, hp.d_idx[b], units * 4, cudaMemcpyDeviceToHost, hp.st[2])) != cudaSuccess) return drained(cuda_fail(e, "D2H idx"));
        cudaEventRecord(hp.ev_out[b], hp.st[2]);
        done += ne; ++it;
    }
    for (int i = 0; i < 3; ++i)
        if ((e = cudaStreamSynchronize(hp.st[i])) != cudaSuccess) return cuda_fail(e, "host pipeline synchronise");
    return AERA_OK;
}

aera_status_t aera_unfold_batch_host(aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                                     int n_samples, double fs_hz, const void *traces_host,
                                     const double *dirs_host, void *efield_host, void *peak_amp_host,
                                     int32_t *peak_idx_host)
{
    return host_impl(pattern, dtype, n_events, n_stations, n_samples, fs_hz, traces_host, 0, nullptr, dirs_host, efield_host,
                     peak_amp_host, peak_idx_host);
}

aera_status_t aera_unfold_batch_host_i16(aera_pattern_t *pattern, int n_events, int n_stations, int n_samples, double fs_hz,
                                         const int16_t *traces_host, const double *counts_to_volts, const double *dirs_host,
                                         float *efield_host, float *peak_amp_host, int32_t *peak_idx_host)
{
    if (!counts_to_volts || !std::isfinite(counts_to_volts[0]) || !std::isfinite(counts_to_volts[1]))
        return fail(AERA_ERR_INVALID_ARG, "counts_to_volts must point to two finite factors (host memory)");
    return host_impl(pattern, AERA_F32, n_events, n_stations, n_samples, fs_hz, traces_host, 1, counts_to_volts, dirs_host, efield_host,
                     peak_amp_host, peak_idx_host);
}

} // extern "C"

// ---- set-up call and hooks of aera_unfold_batch_static (unfold_static.cu)
namespace aera {
aera_status_t report_error(aera_status_t st, const char *msg) { return fail(st, "%s", msg); }
bool plan_is_cached(const aera_pattern_t *pattern, int n_samples, double fs_hz)
{
    aera_pattern *pat = const_cast<aera_pattern *>(pattern);
    std::lock_guard<std::mutex> lk(pat->mu);
    return pat->plans.find(std::make_pair((long long)n_samples | (1LL << 32), fs_hz)) != pat->plans.end();
}
} // namespace aera

extern "C" aera_status_t aera_pattern_prepare(aera_pattern_t *pattern, int n_samples, double fs_hz, void *cuda_stream)
{
    if (!pattern) return fail(AERA_ERR_INVALID_ARG, "pattern is NULL");
    aera_status_t st = check_n(n_samples);
    if (st != AERA_OK) return st;
    Plan *pl = nullptr;
    return get_plan(pattern, n_samples, fs_hz, static_cast<cudaStream_t>(cuda_stream), &pl);
}

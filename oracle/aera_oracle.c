/*
 * aera_oracle.c -- CPU ORACLE for the per-station E-field unfolding of
 * arXiv 1507.07733 ("Prospects of GPGPU in the Auger Offline Software
 * Framework"), section 2 (L29), section 3 (L43-45), section 4 (L59-63, L71).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load it.  It shares no code, header, table or constant with the CUDA
 * path under paper_1507_07733_b200/csrc/.
 *
 * What it is: the plain definition of what the path computes, in IEEE double,
 * with naive O(N*K) discrete Fourier sums (no FFT, no factorisation, no
 * fusion), written in the order of the paper's description:
 *
 *   O1  forward DFT of both channel voltage traces
 *   O2  band selection: bins outside the table band -> 0    (BASELINE north_star)
 *   O3  antenna pattern H_cp(theta,phi,f_k): 8-corner trilinear interpolation of
 *       the tabulated complex VEL, Re and Im independently
 *   O4  per-bin 2x2 complex solve  V = H E
 *   O5  analytic signal: z[n] = (2/N) sum_k E[k] e^{+2 pi i nk/N}
 *   O6  E-field trace e[n] = Re z[n]
 *   O7  Hilbert envelope sqrt(|z_theta|^2+|z_phi|^2), its maximum and the
 *       smallest index attaining it
 *
 * The Fourier sums are accumulated PLAINLY, term after term in index order, not pairwise or compensated (SURVEY.md
 * 8(c) suggested the latter): the error of a plain sum of n terms in double is at most about n * 1.1e-16 relative to
 * the sum of magnitudes, i.e. <= 7e-12 at n = 65536 and <= 5e-13 at n = 4096 in the worst case and about sqrt(n) *
 * 1.1e-16 (3e-14, 7e-15) in practice, well inside the 1e-11 tolerance of the fp64 parity tests; the numpy.fft pins
 * (<= 1e-12) bound it from outside. Keeping the sum plain keeps the function readable against the definition.
 *
 * Readings of the paper where it is silent or garbled are listed in DESIGN.md
 * (section "Readings"); the ones that matter here: envelope = modulus of the analytic
 * signal (R1), forward kernel e^{-2 pi i nk/N} unnormalised, inverse 1/N (R5),
 * DC and Nyquist bins always zero (R4), band edges inclusive (R3),
 * det == 0 -> bin zeroed (R8), zenith clamped / azimuth wrapped (R12, R7).
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"):
 *   O1     numpy.fft on N<=64 and N=256, delta and cosine closed forms, Parseval
 *   O2     band limits of the five BASELINE configs (tests/golden/band_limits.txt)
 *   O3     exact at grid nodes, multilinear functions reproduced, cell centre =
 *          mean of 8 corners, azimuth periodicity, scipy RegularGridInterpolator
 *   O4     numpy.linalg.solve
 *   O4+O5  fold -> unfold round trip <= 1e-10 (on-node and off-node)
 *   O1-O7  H == identity reduces to brick-wall band-pass + scipy.signal.hilbert
 *   O5-O7  in-band cosine -> constant envelope A; synthetic pulse -> (A, n0)
 * Conventions with nothing in the paper to pin them (R4 DC/Nyquist, R8 singular
 * H, R12 zenith clamp) are unit-tested as conventions only: "parity unpinned"
 * for those three corner behaviours.
 *
 * Build:  gcc -O2 -fopenmp -fPIC -shared -o liboracle_aera.so aera_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int n_zenith;
    double zenith0_deg, dzenith_deg;
    int n_azimuth;
    double azimuth0_deg, dazimuth_deg;
    int azimuth_periodic;
    int n_freq;
    double freq0_hz, dfreq_hz;
} oracle_grid_t;

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* W[m] = exp(-2 pi i m / N), m = 0..N-1, evaluated in long double, rounded once. */
void oracle_twiddles(int N, double *Wre, double *Wim)
{
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int m = 0; m < N; ++m) {
        long double a = two_pi * (long double)m / (long double)N;
        Wre[m] = (double)cosl(a);
        Wim[m] = (double)(-sinl(a));
    }
}

/* O2: k_lo = smallest k with f0 <= k fs/N, k_hi = largest k with k fs/N <= f_hi,
 * both additionally confined to 1 .. N/2-1 (DC and Nyquist never in band).
 * The comparison f0*N <= k*fs is made exactly when fs, f0, df are integers (Hz). */
static int is_integral(double x) { return x == floor(x) && fabs(x) < 9.0e15; }

void oracle_band(int N, double fs_hz, int n_freq, double freq0_hz, double dfreq_hz,
                 long *k_lo, long *k_hi)
{
    long lo = N, hi = -1;
    const int exact = is_integral(fs_hz) && is_integral(freq0_hz) && is_integral(dfreq_hz);
    for (long k = 1; k < N / 2; ++k) {
        int in;
        if (exact) {
            __int128 kfs = (__int128)k * (__int128)(long long)fs_hz;
            __int128 lo_n = (__int128)(long long)freq0_hz * N;
            __int128 hi_n = ((__int128)(long long)freq0_hz +
                             (__int128)(n_freq - 1) * (__int128)(long long)dfreq_hz) * N;
            in = (kfs >= lo_n) && (kfs <= hi_n);
        } else {
            long double f = (long double)k * (long double)fs_hz / (long double)N;
            long double fhi = (long double)freq0_hz + (long double)(n_freq - 1) * (long double)dfreq_hz;
            in = (f >= (long double)freq0_hz) && (f <= fhi);
        }
        if (in) {
            if (k < lo) lo = k;
            if (k > hi) hi = k;
        }
    }
    *k_lo = lo;
    *k_hi = hi; /* empty band: lo = N > hi = -1 */
}

/* O1: X[k - k_lo] = sum_n x[n] W[(n k) mod N], k = k_lo..k_hi.  The index n*k is
 * reduced mod N in integers (incrementally), never as a floating argument. */
void oracle_dft_band(const double *x, int N, long k_lo, long k_hi,
                     const double *Wre, const double *Wim, double *Xre, double *Xim)
{
    for (long k = k_lo; k <= k_hi; ++k) {
        double sr = 0.0, si = 0.0;
        long m = 0;
        for (int n = 0; n < N; ++n) {
            sr += x[n] * Wre[m];
            si += x[n] * Wim[m];
            m += k;
            if (m >= N) m -= N;
        }
        Xre[k - k_lo] = sr;
        Xim[k - k_lo] = si;
    }
}

/* Fractional coordinate -> (cell index, weight) on a uniform axis of n nodes.
 * i = min(floor(u), n-2), t = u - i, so the upper edge gives t = 1. */
static void cell_of(double u, int n, int *i, double *t)
{
    double fl = floor(u);
    int ii = (int)fl;
    if (ii > n - 2) ii = n - 2;
    if (ii < 0) ii = 0;
    *i = ii;
    *t = u - (double)ii;
}

/* O3: H_cp(theta, phi, f) by 8-corner trilinear interpolation.
 * H is [2][2][n_z][n_a][n_f] interleaved (re, im) doubles.  out = {H0t, H0p, H1t, H1p}
 * as (re, im) pairs.  Zenith clamped to the table, azimuth wrapped to one period
 * (periodic axis: the stored last node duplicates the first and is never read),
 * frequency clamped (callers only ask for in-band frequencies). */
void oracle_pattern_eval(const oracle_grid_t *g, const double *H,
                         double theta_deg, double phi_deg, double f_hz, double out[8])
{
    const int nz = g->n_zenith, na = g->n_azimuth, nf = g->n_freq;
    double zmax = g->zenith0_deg + (nz - 1) * g->dzenith_deg;
    double th = theta_deg;
    if (th < g->zenith0_deg) th = g->zenith0_deg;
    if (th > zmax) th = zmax;
    double uz = (th - g->zenith0_deg) / g->dzenith_deg;
    int iz; double tz;
    cell_of(uz, nz, &iz, &tz);

    int ia, ia1; double ta;
    if (g->azimuth_periodic) {
        double P = (na - 1) * g->dazimuth_deg;
        double pw = phi_deg - P * floor((phi_deg - g->azimuth0_deg) / P);
        double ua = (pw - g->azimuth0_deg) / g->dazimuth_deg;
        double fl = floor(ua);
        ia = (int)fl;
        if (ia >= na - 1) ia -= (na - 1); /* pw == a0 + P by rounding */
        if (ia < 0) ia = 0;
        ta = ua - fl;
        ia1 = (ia + 1) % (na - 1);
    } else {
        double amax = g->azimuth0_deg + (na - 1) * g->dazimuth_deg;
        double p = phi_deg;
        if (p < g->azimuth0_deg) p = g->azimuth0_deg;
        if (p > amax) p = amax;
        cell_of((p - g->azimuth0_deg) / g->dazimuth_deg, na, &ia, &ta);
        ia1 = ia + 1;
    }

    double fmax = g->freq0_hz + (nf - 1) * g->dfreq_hz;
    double f = f_hz;
    if (f < g->freq0_hz) f = g->freq0_hz;
    if (f > fmax) f = fmax;
    int jf; double tf;
    cell_of((f - g->freq0_hz) / g->dfreq_hz, nf, &jf, &tf);

    const int zi[2] = { iz, iz + 1 };
    const int ai[2] = { ia, ia1 };
    const double wz[2] = { 1.0 - tz, tz };
    const double wa[2] = { 1.0 - ta, ta };
    const double wf[2] = { 1.0 - tf, tf };
    for (int cp = 0; cp < 4; ++cp) {
        double re = 0.0, im = 0.0;
        for (int dz = 0; dz < 2; ++dz)
            for (int da = 0; da < 2; ++da)
                for (int dfi = 0; dfi < 2; ++dfi) {
                    size_t idx = ((((size_t)cp * nz + zi[dz]) * na + ai[da]) * nf + (jf + dfi));
                    double w = wz[dz] * wa[da] * wf[dfi];
                    re += w * H[2 * idx];
                    im += w * H[2 * idx + 1];
                }
        out[2 * cp] = re;
        out[2 * cp + 1] = im;
    }
}

static void cmul(double ar, double ai, double br, double bi, double *cr, double *ci)
{
    *cr = ar * br - ai * bi;
    *ci = ar * bi + ai * br;
}

/* O4: solve V = H E for E.  h = {H0t, H0p, H1t, H1p}, v = {V0, V1}, e = {Et, Ep},
 * all (re, im).  det == 0 -> E = 0, returns 0; else 1. */
int oracle_solve2x2(const double h[8], const double v[4], double e[4])
{
    double d1r, d1i, d2r, d2i;
    cmul(h[0], h[1], h[6], h[7], &d1r, &d1i); /* H0t*H1p */
    cmul(h[2], h[3], h[4], h[5], &d2r, &d2i); /* H0p*H1t */
    double dr = d1r - d2r, di = d1i - d2i;
    double den = dr * dr + di * di;
    if (den == 0.0) { e[0] = e[1] = e[2] = e[3] = 0.0; return 0; }
    double ar, ai, br, bi, nr, ni;
    /* Et = (H1p V0 - H0p V1)/det */
    cmul(h[6], h[7], v[0], v[1], &ar, &ai);
    cmul(h[2], h[3], v[2], v[3], &br, &bi);
    nr = ar - br; ni = ai - bi;
    e[0] = (nr * dr + ni * di) / den;
    e[1] = (ni * dr - nr * di) / den;
    /* Ep = (H0t V1 - H1t V0)/det */
    cmul(h[0], h[1], v[2], v[3], &ar, &ai);
    cmul(h[4], h[5], v[0], v[1], &br, &bi);
    nr = ar - br; ni = ai - bi;
    e[2] = (nr * dr + ni * di) / den;
    e[3] = (ni * dr - nr * di) / den;
    return 1;
}

/* O5: z[n] = (2/N) sum_{k=k_lo}^{k_hi} E[k-k_lo] conj(W[(n k) mod N]), n = 0..N-1. */
void oracle_analytic_from_band(const double *Ere, const double *Eim, int N, long k_lo, long k_hi,
                               const double *Wre, const double *Wim, double *zre, double *zim)
{
    const double s = 2.0 / (double)N;
    for (int n = 0; n < N; ++n) {
        double sr = 0.0, si = 0.0;
        long m = (long)(((long long)n * (long long)k_lo) % N);
        for (long k = k_lo; k <= k_hi; ++k) {
            double wr = Wre[m], wi = -Wim[m]; /* conj */
            double er = Ere[k - k_lo], ei = Eim[k - k_lo];
            sr += er * wr - ei * wi;
            si += er * wi + ei * wr;
            m += n;
            if (m >= N) m -= N;
        }
        zre[n] = s * sr;
        zim[n] = s * si;
    }
}

/* O7: env2[n] = |zt|^2 + |zp|^2; idx = smallest n attaining max; amp = sqrt(max). */
void oracle_peak(const double *ztre, const double *ztim, const double *zpre, const double *zpim,
                 int N, double *env2_out /* may be NULL */, double *amp, int32_t *idx)
{
    double best = -1.0; int32_t bi = 0;
    for (int n = 0; n < N; ++n) {
        double e2 = ztre[n] * ztre[n] + ztim[n] * ztim[n] + zpre[n] * zpre[n] + zpim[n] * zpim[n];
        if (env2_out) env2_out[n] = e2;
        if (e2 > best) { best = e2; bi = n; }
    }
    *amp = sqrt(best);
    *idx = bi;
}

/* One station, O1..O7.  v = [2][N]; efield = [2][N] (theta, phi); env2 = [N] or NULL.
 * spec_out (may be NULL) receives the band spectra {V0, V1, Et, Ep} as [4][K][2]. */
static void unfold_station(const oracle_grid_t *g, const double *H, int N, double fs_hz,
                           long k_lo, long k_hi, const double *Wre, const double *Wim,
                           const double *v, double theta_deg, double phi_deg,
                           double *efield, double *env2, double *amp, int32_t *idx,
                           double *spec_out)
{
    long K = (k_hi >= k_lo) ? (k_hi - k_lo + 1) : 0;
    double *buf = (double *)calloc((size_t)(8 * (K > 0 ? K : 1) + 4 * (size_t)N), sizeof(double));
    double *V0r = buf, *V0i = V0r + K, *V1r = V0i + K, *V1i = V1r + K;
    double *Etr = V1i + K, *Eti = Etr + K, *Epr = Eti + K, *Epi = Epr + K;
    double *ztr = Epi + K, *zti = ztr + N, *zpr = zti + N, *zpi = zpr + N;

    if (K > 0) {
        oracle_dft_band(v, N, k_lo, k_hi, Wre, Wim, V0r, V0i);     /* O1 channel 0 */
        oracle_dft_band(v + N, N, k_lo, k_hi, Wre, Wim, V1r, V1i); /* O1 channel 1 */
        for (long k = k_lo; k <= k_hi; ++k) {
            double f = (double)k * fs_hz / (double)N;
            double h[8], vv[4], e[4];
            oracle_pattern_eval(g, H, theta_deg, phi_deg, f, h);    /* O3 */
            vv[0] = V0r[k - k_lo]; vv[1] = V0i[k - k_lo];
            vv[2] = V1r[k - k_lo]; vv[3] = V1i[k - k_lo];
            oracle_solve2x2(h, vv, e);                              /* O4 */
            Etr[k - k_lo] = e[0]; Eti[k - k_lo] = e[1];
            Epr[k - k_lo] = e[2]; Epi[k - k_lo] = e[3];
        }
        oracle_analytic_from_band(Etr, Eti, N, k_lo, k_hi, Wre, Wim, ztr, zti); /* O5 */
        oracle_analytic_from_band(Epr, Epi, N, k_lo, k_hi, Wre, Wim, zpr, zpi);
    }
    if (efield)
        for (int n = 0; n < N; ++n) { efield[n] = ztr[n]; efield[N + n] = zpr[n]; } /* O6 */
    oracle_peak(ztr, zti, zpr, zpi, N, env2, amp, idx);                         /* O7 */
    if (spec_out) {
        for (long j = 0; j < K; ++j) {
            spec_out[2 * (0 * K + j)] = V0r[j]; spec_out[2 * (0 * K + j) + 1] = V0i[j];
            spec_out[2 * (1 * K + j)] = V1r[j]; spec_out[2 * (1 * K + j) + 1] = V1i[j];
            spec_out[2 * (2 * K + j)] = Etr[j]; spec_out[2 * (2 * K + j) + 1] = Eti[j];
            spec_out[2 * (3 * K + j)] = Epr[j]; spec_out[2 * (3 * K + j) + 1] = Epi[j];
        }
    }
    free(buf);
}

/* Batch of independent units.  traces [n_units][2][N], dirs [n_units][2] (zenith, azimuth
 * in degrees; the caller repeats the event direction for each of its stations),
 * efield [n_units][2][N] or NULL, env2 [n_units][N] or NULL, amp/idx [n_units].
 * OpenMP over units. Returns the number of in-band bins K. */
long oracle_unfold_batch(const oracle_grid_t *g, const double *H, long n_units, int N, double fs_hz,
                         const double *traces, const double *dirs,
                         double *efield, double *env2, double *amp, int32_t *idx)
{
    long k_lo, k_hi;
    oracle_band(N, fs_hz, g->n_freq, g->freq0_hz, g->dfreq_hz, &k_lo, &k_hi);
    double *Wre = (double *)malloc(sizeof(double) * (size_t)N);
    double *Wim = (double *)malloc(sizeof(double) * (size_t)N);
    oracle_twiddles(N, Wre, Wim);
#pragma omp parallel for schedule(dynamic, 1)
    for (long u = 0; u < n_units; ++u) {
        unfold_station(g, H, N, fs_hz, k_lo, k_hi, Wre, Wim,
                       traces + (size_t)u * 2 * N, dirs[2 * u], dirs[2 * u + 1],
                       efield ? efield + (size_t)u * 2 * N : NULL,
                       env2 ? env2 + (size_t)u * N : NULL, amp + u, idx + u, NULL);
    }
    free(Wre); free(Wim);
    return (k_hi >= k_lo) ? (k_hi - k_lo + 1) : 0;
}

/* Single station, also returning the band spectra {V0,V1,Et,Ep} [4][K] complex. */
long oracle_unfold_station_spectra(const oracle_grid_t *g, const double *H, int N, double fs_hz,
                                   const double *v, double theta_deg, double phi_deg,
                                   double *efield, double *env2, double *amp, int32_t *idx,
                                   double *spec_out)
{
    long k_lo, k_hi;
    oracle_band(N, fs_hz, g->n_freq, g->freq0_hz, g->dfreq_hz, &k_lo, &k_hi);
    double *Wre = (double *)malloc(sizeof(double) * (size_t)N);
    double *Wim = (double *)malloc(sizeof(double) * (size_t)N);
    oracle_twiddles(N, Wre, Wim);
    unfold_station(g, H, N, fs_hz, k_lo, k_hi, Wre, Wim, v, theta_deg, phi_deg,
                   efield, env2, amp, idx, spec_out);
    free(Wre); free(Wim);
    return (k_hi >= k_lo) ? (k_hi - k_lo + 1) : 0;
}

/* Direction scan (BASELINE configs[2]): O1 once per station, O3-O7 for every direction.
 * traces [S][2][N]; dirs [D][2]; amp, idx [D][S]; env2 [D][S][N] or NULL (the squared envelope
 * of every pair, so that a test can apply the near-tie rule of BASELINE north_star: "+-1 allowed when
 * the top two envelope values differ by < 1e-5 relative").  OpenMP over (direction, station). */
long oracle_scan(const oracle_grid_t *g, const double *H, int S, int N, double fs_hz,
                 const double *traces, long D, const double *dirs, double *amp, int32_t *idx,
                 double *env2)
{
    long k_lo, k_hi;
    oracle_band(N, fs_hz, g->n_freq, g->freq0_hz, g->dfreq_hz, &k_lo, &k_hi);
    long K = (k_hi >= k_lo) ? (k_hi - k_lo + 1) : 0;
    double *Wre = (double *)malloc(sizeof(double) * (size_t)N);
    double *Wim = (double *)malloc(sizeof(double) * (size_t)N);
    oracle_twiddles(N, Wre, Wim);
    size_t KK = (size_t)(K > 0 ? K : 1);
    double *V = (double *)calloc((size_t)S * 4 * KK, sizeof(double)); /* [S]{V0r,V0i,V1r,V1i}[K] */
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < S; ++s) {
        double *b = V + (size_t)s * 4 * KK;
        if (K > 0) {
            oracle_dft_band(traces + (size_t)s * 2 * N, N, k_lo, k_hi, Wre, Wim, b, b + KK);
            oracle_dft_band(traces + (size_t)s * 2 * N + N, N, k_lo, k_hi, Wre, Wim, b + 2 * KK, b + 3 * KK);
        }
    }
#pragma omp parallel for schedule(dynamic, 1)
    for (long p = 0; p < D * (long)S; ++p) {
        long d = p / S; int s = (int)(p % S);
        const double *b = V + (size_t)s * 4 * KK;
        double *w = (double *)calloc(4 * KK + 4 * (size_t)N, sizeof(double));
        double *Etr = w, *Eti = Etr + KK, *Epr = Eti + KK, *Epi = Epr + KK;
        double *ztr = Epi + KK, *zti = ztr + N, *zpr = zti + N, *zpi = zpr + N;
        for (long k = k_lo; k <= k_hi; ++k) {
            long j = k - k_lo;
            double f = (double)k * fs_hz / (double)N;
            double h[8], vv[4], e[4];
            oracle_pattern_eval(g, H, dirs[2 * d], dirs[2 * d + 1], f, h);
            vv[0] = b[j]; vv[1] = b[KK + j]; vv[2] = b[2 * KK + j]; vv[3] = b[3 * KK + j];
            oracle_solve2x2(h, vv, e);
            Etr[j] = e[0]; Eti[j] = e[1]; Epr[j] = e[2]; Epi[j] = e[3];
        }
        if (K > 0) {
            oracle_analytic_from_band(Etr, Eti, N, k_lo, k_hi, Wre, Wim, ztr, zti);
            oracle_analytic_from_band(Epr, Epi, N, k_lo, k_hi, Wre, Wim, zpr, zpi);
        }
        oracle_peak(ztr, zti, zpr, zpi, N, env2 ? env2 + (size_t)p * N : NULL, amp + p, idx + p);
        free(w);
    }
    free(V); free(Wre); free(Wim);
    return K;
}

/* Forward model (test helper; inverse of O4 followed by the inverse real DFT):
 * band spectra Et, Ep [K] complex -> V_c[k] = H_ct E_t + H_cp E_p, then
 * v_c[n] = (1/N) * 2 Re sum_k V_c[k] e^{+2 pi i nk/N}.  v = [2][N]. */
long oracle_fold_station(const oracle_grid_t *g, const double *H, int N, double fs_hz,
                         const double *Et /*[K][2]*/, const double *Ep /*[K][2]*/,
                         double theta_deg, double phi_deg, double *v)
{
    long k_lo, k_hi;
    oracle_band(N, fs_hz, g->n_freq, g->freq0_hz, g->dfreq_hz, &k_lo, &k_hi);
    long K = (k_hi >= k_lo) ? (k_hi - k_lo + 1) : 0;
    double *Wre = (double *)malloc(sizeof(double) * (size_t)N);
    double *Wim = (double *)malloc(sizeof(double) * (size_t)N);
    oracle_twiddles(N, Wre, Wim);
    size_t KK = (size_t)(K > 0 ? K : 1);
    double *V = (double *)calloc(4 * KK, sizeof(double));
    for (long k = k_lo; k <= k_hi; ++k) {
        long j = k - k_lo;
        double f = (double)k * fs_hz / (double)N;
        double h[8], ar, ai, br, bi;
        oracle_pattern_eval(g, H, theta_deg, phi_deg, f, h);
        cmul(h[0], h[1], Et[2 * j], Et[2 * j + 1], &ar, &ai);
        cmul(h[2], h[3], Ep[2 * j], Ep[2 * j + 1], &br, &bi);
        V[j] = ar + br; V[KK + j] = ai + bi;
        cmul(h[4], h[5], Et[2 * j], Et[2 * j + 1], &ar, &ai);
        cmul(h[6], h[7], Ep[2 * j], Ep[2 * j + 1], &br, &bi);
        V[2 * KK + j] = ar + br; V[3 * KK + j] = ai + bi;
    }
    for (int c = 0; c < 2; ++c)
        for (int n = 0; n < N; ++n) {
            double sr = 0.0;
            long m = (K > 0) ? (long)(((long long)n * (long long)k_lo) % N) : 0;
            for (long k = k_lo; k <= k_hi; ++k) {
                long j = k - k_lo;
                /* Re( V * conj(W) ) */
                sr += V[2 * c * KK + j] * Wre[m] + V[(2 * c + 1) * KK + j] * Wim[m];
                m += n;
                if (m >= N) m -= N;
            }
            v[(size_t)c * N + n] = 2.0 * sr / (double)N;
        }
    free(V); free(Wre); free(Wim);
    return K;
}

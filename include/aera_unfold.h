/*
 * aera_unfold.h -- C ABI of the B200-native per-station E-field unfolding library
 * (libaera_unfold.so), the data-parallel hot path of the AERA radio reconstruction of
 * arXiv 1507.07733.
 *
 * The operation (section 2: "the antenna pattern for this direction is evaluated,
 * and the E-field trace at each station reconstructed from the voltage traces. Finally, the
 * maximum of the envelope of the E-field trace is used as updated timing information";
 * section 3: vector effective length tabulated on (frequency, zenith, azimuth) nodes and
 * interpolated linearly; section 4, L59-63 and L71: Fourier transforms and the Hilbert envelope):
 *
 *   for every station of every event, with the event's shower direction (theta, phi):
 *     V_c[k]  = sum_n v_c[n] exp(-2 pi i n k / N)              c = 0,1  (forward real DFT)
 *     H_cp[k] = trilinear interpolation of the tabulated complex response at
 *               (theta, phi, f_k = k fs / N); azimuth periodic; bins outside the table
 *               band, DC and Nyquist are zeroed
 *     E[k]    = H[k]^-1 V[k]                                   (2x2 complex solve, p = theta,phi)
 *     z_p[n]  = (2/N) sum_{k in band} E_p[k] exp(+2 pi i n k / N)   (analytic signal)
 *     e_p[n]  = Re z_p[n]                                      (E-field traces)
 *     env[n]  = sqrt(|z_theta[n]|^2 + |z_phi[n]|^2)            (Hilbert envelope)
 *     peak_amp = max_n env[n], peak_idx = smallest n attaining it
 *
 * All entry points are plain C: pointers (host or device as stated per argument), sizes,
 * and an opaque CUDA stream handle (cudaStream_t passed as void*; NULL = legacy default
 * stream).  No exceptions cross the ABI; every call returns an aera_status_t and sets a
 * thread-local message readable with aera_last_error().
 *
 * Unless stated otherwise calls are ASYNCHRONOUS on the given stream: they validate their
 * arguments on the host, enqueue kernels, and return without synchronising.  They allocate
 * nothing on the hot path: scratch memory is caller-provided (aera_workspace_bytes).  The only
 * allocations the library makes are (a) inside aera_pattern_upload, (b) the first time a
 * pattern is used with a new (n_samples, fs_hz) pair, when a small plan (twiddle tables,
 * per-bin frequency cell/weight table) is built and cached in the pattern handle -- that first
 * call synchronises the stream once -- and (c) inside the *_host convenience entry point.
 */
#ifndef AERA_UNFOLD_H
#define AERA_UNFOLD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct aera_pattern aera_pattern_t; /* opaque; owns the device copy of one table + plans */

typedef enum { AERA_F32 = 0, AERA_F64 = 1 } aera_dtype_t;

typedef enum {
    AERA_OK = 0,
    AERA_ERR_INVALID_ARG = 1,   /* NULL pointer, non-positive size, misaligned buffer, bad grid */
    AERA_ERR_UNSUPPORTED_N = 2, /* n_samples not a power of two in [64, 65536] */
    AERA_ERR_DTYPE_MISMATCH = 3,/* dtype differs from the pattern's dtype */
    AERA_ERR_WORKSPACE = 4,     /* workspace NULL/misaligned/smaller than aera_workspace_bytes() */
    AERA_ERR_ALLOC = 5,         /* cudaMalloc / host allocation failed */
    AERA_ERR_CUDA = 6,          /* a CUDA runtime call or launch failed; message has the string */
    AERA_ERR_BAND = 7           /* table band does not lie inside (0, fs/2) or contains no bin */
} aera_status_t;

/* Uniform node grids. Angles in DEGREES, frequency in Hz ("discrete frequencies and
 * zenith and azimuth angles").  When azimuth_periodic != 0 the axis has period
 * (n_azimuth-1)*dazimuth_deg and the stored last node must duplicate the first; the library never
 * reads the last node and wraps instead.  Zenith outside the table is clamped to the table. */
typedef struct {
    int dtype;              /* AERA_F32: complex64 table; AERA_F64: complex128 table */
    int n_zenith;  double zenith0_deg,  dzenith_deg;    /* >= 2 nodes, step > 0 */
    int n_azimuth; double azimuth0_deg, dazimuth_deg;   /* >= 2 nodes (>= 3 if periodic), step > 0 */
    int azimuth_periodic;
    int n_freq;    double freq0_hz, dfreq_hz;           /* 2 <= n_freq <= 512, step > 0 */
} aera_pattern_desc_t;

/* Copy one antenna-response table to the device and repack it (once) into the library's
 * layout [zenith][azimuth][freq][channel*2+pol] ("the patterns are copied and
 * converted ... only once on first access").
 *   H    interleaved (re, im), C order [channel 2][pol 2 (theta,phi)][n_zenith][n_azimuth][n_freq],
 *        element type complex64 or complex128 per desc->dtype.  HOST pointer if
 *        src_on_device == 0, DEVICE pointer otherwise.  Not retained: the caller may free it
 *        after the call returns (the call synchronises the stream before returning).
 *   out  receives the handle; release with aera_pattern_free. Several patterns may be resident.
 * Errors: INVALID_ARG (NULL, bad grid), ALLOC, CUDA. */
aera_status_t aera_pattern_upload(const aera_pattern_desc_t *desc, const void *H, int src_on_device,
                                  void *cuda_stream, aera_pattern_t **out);

/* Frees the device table and all cached plans. The caller guarantees no kernel using it is in
 * flight. NULL is accepted. */
aera_status_t aera_pattern_free(aera_pattern_t *pattern);

/* In-band DFT bins for (pattern, n_samples, fs_hz): k_lo..k_hi inclusive, the bins with
 * freq0 <= k*fs/N <= freq0+(n_freq-1)*dfreq and 0 < k < N/2 (evaluated exactly in integers when
 * fs, freq0, dfreq are whole numbers of Hz).  Errors: UNSUPPORTED_N, BAND. */
aera_status_t aera_band(const aera_pattern_t *pattern, int n_samples, double fs_hz,
                        int *k_lo, int *k_hi);

typedef enum { AERA_OP_UNFOLD = 0, AERA_OP_SCAN = 1, AERA_OP_FOLD = 2, AERA_OP_RECONSTRUCT = 3 } aera_op_t;

/* Scratch bytes needed by aera_unfold_batch (n_events_or_dirs = n_events) or
 * aera_scan_directions (n_events_or_dirs = n_dirs) for these sizes; 0 on invalid arguments
 * (aera_last_error tells why).  The workspace holds the per-event (per-direction) inverse
 * response matrices and, for the kernels that need it, per-CTA transform buffers / per-station
 * spectra.  Contents are undefined between calls; one workspace must not be shared by calls
 * that may run concurrently. */
size_t aera_workspace_bytes(aera_op_t op, const aera_pattern_t *pattern, int dtype,
                            long n_events_or_dirs, int n_stations, int n_samples, double fs_hz);

/* Batched unfolding (PAPER.md L29 step 3+4 for every station of every event).
 *   traces    DEVICE [n_events][n_stations][2 channels][n_samples] real (dtype), 16-byte aligned
 *   dirs      DEVICE [n_events][2] double: (zenith_deg, azimuth_deg), one direction per event
 *   efield    DEVICE [n_events][n_stations][2 (theta,phi)][n_samples] real (dtype), 16-byte aligned;
 *             may be the same pointer as traces (in place); may be NULL (peaks only)
 *   peak_amp  DEVICE [n_events][n_stations] real (dtype)     envelope maximum
 *   peak_idx  DEVICE [n_events][n_stations] int32            smallest sample index attaining it
 *   workspace DEVICE, 256-byte aligned, >= aera_workspace_bytes(AERA_OP_UNFOLD, ...)
 * All buffers are caller-owned. n_samples: power of two in [64, 65536]. The result is linear in
 * the traces; units are the caller's (configs: microvolt in, microvolt/metre out).
 * NaN/Inf in the data are not checked (they propagate). n_events == 0 is a no-op.
 * No call changes device-wide state unless asked to (aera_set_long_trace_l2_persist below is the one request there is).
 * Errors: INVALID_ARG, UNSUPPORTED_N, DTYPE_MISMATCH, WORKSPACE, BAND, ALLOC (first-use plan), CUDA. */
aera_status_t aera_unfold_batch(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                                int n_samples, double fs_hz, const void *traces, const double *dirs,
                                void *efield, void *peak_amp, int32_t *peak_idx,
                                void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Direction-hypothesis scan (BASELINE configs[2]; motivated by PAPER.md L29: the pattern is
 * re-evaluated at a new direction in every iteration of the reconstruction loop): one forward
 * transform per station, then unfolding + envelope peak at every direction; no trace output.
 *   traces    DEVICE [n_stations][2][n_samples] real (dtype), 16-byte aligned
 *   dirs      DEVICE [n_dirs][2] double (zenith_deg, azimuth_deg)
 *   peak_amp  DEVICE [n_dirs][n_stations] real (dtype);  peak_idx DEVICE [n_dirs][n_stations] int32
 *   workspace DEVICE, 256-byte aligned, >= aera_workspace_bytes(AERA_OP_SCAN, ..., n_dirs, ...)
 * Errors as aera_unfold_batch. */
aera_status_t aera_scan_directions(const aera_pattern_t *pattern, int dtype, int n_stations,
                                   int n_samples, double fs_hz, const void *traces,
                                   long n_dirs, const double *dirs,
                                   void *peak_amp, int32_t *peak_idx,
                                   void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * Optional pre-filter fused into the unfolding (section 2: "noise filtering and signal
 * enhancing" precedes the loop; the paper does not specify the filter). One real weight per in-band DFT
 * bin k_lo .. k_hi of a given (n_samples, fs_hz) (aera_band gives the range; n_weights must equal
 * k_hi - k_lo + 1): E[k] = weights[k - k_lo] * H[k]^-1 V[k], e.g. a band-pass taper or notches at narrow-band
 * transmitters. The weights are folded into the per-direction matrices, so the filter costs nothing per
 * station. It applies to aera_unfold_batch, aera_scan_directions and aera_reconstruct_batch of this pattern
 * for that (n_samples, fs_hz) until replaced; weights == NULL removes it. The multi-table, int16 and up-sampled
 * variants apply it too (up-sampling does not change the band: z[upsample * n] stays sample n of the filtered
 * aera_unfold_batch). aera_fold_batch ignores it.
 * weights is a HOST pointer. A configuration call, not a hot one: it synchronises the whole DEVICE (no kernel of an
 * earlier call on any stream may still be reading the old weights) and then the stream for the upload.
 */
aera_status_t aera_pattern_set_band_filter(aera_pattern_t *pattern, int n_samples, double fs_hz, const double *weights,
                                           int n_weights, void *cuda_stream);

/*
 * Forward model on the device (the inverse of the solve of aera_unfold_batch; section 3: the
 * voltage of each channel is the vector effective length applied to the electric field vector): for every
 * station, with the event's direction,
 *     E_p[k]  = sum_n e_p[n] exp(-2 pi i n k / N),  p = theta, phi
 *     V_c[k]  = H_c,theta[k] E_theta[k] + H_c,phi[k] E_phi[k]   on the table band, 0 elsewhere (and at DC, Nyquist)
 *     v_c[n]  = (2/N) Re sum_{k in band} V_c[k] exp(+2 pi i n k / N)
 * i.e. the band-limited E-field folded with the interpolated antenna response. It runs the same fused
 * kernels as aera_unfold_batch with the matrix (1/N) H in place of (1/N) H^-1.
 *   efield [n_events][n_stations][2 (theta, phi)][n_samples] real, device, in
 *   dirs   [n_events][2] double degrees, device
 *   traces [n_events][n_stations][2 (channels)][n_samples] real, device, out; may alias efield
 *   workspace >= aera_workspace_bytes(AERA_OP_FOLD, ...)
 */
aera_status_t aera_fold_batch(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                              int n_samples, double fs_hz, const void *efield, const double *dirs,
                              void *traces, void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * Several pattern tables, one antenna type per station (section 3: "The patterns for all antennas used in
 * AERA can be stored simultaneously on the device"; L43: "For each antenna, the VEL is known for discrete frequencies and
 * zenith and azimuth angles"). Exactly aera_unfold_batch, except that station s of every event is unfolded with the table
 * patterns[pattern_id[s]]; the per-direction matrices are then built once per (event, table).
 *   patterns    HOST array of n_patterns handles (1..64), all of the call's dtype and with the same frequency axis
 *               (n_freq, freq0_hz, dfreq_hz: the in-band bins must agree); zenith / azimuth grids may differ
 *   pattern_id  DEVICE [n_stations] int32, values in 0 .. n_patterns-1. The call is asynchronous and the array is on the
 *               device, so a value outside that range cannot be reported: it is clamped to the nearest valid table
 *               (a negative id uses table 0, a too large one the last table) and never indexes outside the workspace
 *   workspace   >= aera_workspace_bytes_ex(AERA_OP_UNFOLD, patterns[0], dtype, n_events, n_stations, n_samples, fs_hz,
 *               n_patterns, 1)
 * A band filter set on patterns[0] applies to all tables. Errors as aera_unfold_batch.
 */
aera_status_t aera_unfold_batch_multi(const aera_pattern_t *const *patterns, int n_patterns, const int32_t *pattern_id,
                                      int dtype, int n_events, int n_stations, int n_samples, double fs_hz,
                                      const void *traces, const double *dirs, void *efield, void *peak_amp, int32_t *peak_idx,
                                      void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * int16 ADC-count input (section 2: "the voltage traces of the two channels at each station are read out";
 * the station electronics deliver ADC counts, the paper does not give the conversion). The traces are read as int16, which
 * halves the bytes read per station (24 584 algorithmic bytes per unit at n_samples = 2048 instead of 32 776):
 *     v_c[n] = counts_to_volts[c] * traces[..][c][n]       then exactly aera_unfold_batch in fp32
 * (the two factors are folded into the per-direction matrices: the unfolding is linear in the traces).
 *   traces           DEVICE [n_events][n_stations][2][n_samples] int16, 16-byte aligned
 *   counts_to_volts  HOST [2] double, one factor per channel
 *   efield / peak_amp / peak_idx  as aera_unfold_batch with dtype AERA_F32 (efield cannot alias traces)
 *   pattern          an AERA_F32 pattern; workspace >= aera_workspace_bytes(AERA_OP_UNFOLD, pattern, AERA_F32, ...)
 */
aera_status_t aera_unfold_batch_i16(const aera_pattern_t *pattern, int n_events, int n_stations, int n_samples, double fs_hz,
                                    const int16_t *traces, const double *counts_to_volts, const double *dirs,
                                    float *efield, float *peak_amp, int32_t *peak_idx,
                                    void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * Spectral up-sampling by zero-padding (section 2: "after noise filtering and signal enhancing"; the paper
 * does not specify the enhancement, reading R23): the unfolded band spectrum is unchanged and the analytic signal
 * is evaluated on a grid `upsample` times finer,
 *     z_p[n] = (2/N) sum_{k in band} E_p[k] exp(+2 pi i n k / (upsample N)),   n = 0 .. upsample N - 1,
 * so that z[upsample n] is the sample n of aera_unfold_batch and the envelope maximum is found with sub-sample timing.
 *   upsample  power of two >= 1 with upsample * n_samples <= 65536
 *   efield    DEVICE [n_events][n_stations][2][upsample * n_samples] (may be NULL; cannot alias traces unless upsample == 1)
 *   peak_idx  index on the FINE grid (0 .. upsample * n_samples - 1), peak_amp the envelope maximum there
 *   workspace >= aera_workspace_bytes_ex(AERA_OP_UNFOLD, pattern, dtype, n_events, n_stations, n_samples, fs_hz, 1, upsample)
 * upsample > 1 runs on the generic kernels (aera_last_kernel() says so).
 */
aera_status_t aera_unfold_batch_upsampled(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations, int n_samples,
                                          double fs_hz, int upsample, const void *traces, const double *dirs,
                                          void *efield, void *peak_amp, int32_t *peak_idx,
                                          void *workspace, size_t workspace_bytes, void *cuda_stream);

/* aera_workspace_bytes for the calls above: n_patterns tables (1 for a single one), spectral up-sampling factor (1 = none). */
size_t aera_workspace_bytes_ex(aera_op_t op, const aera_pattern_t *pattern, int dtype, long n_events_or_dirs,
                               int n_stations, int n_samples, double fs_hz, int n_patterns, int upsample);

/*
 * Device-resident reconstruction loop (section 2, L29 and Fig. 1: "First, as an initial estimate of the
 * event timing in each station, the maxima of the voltage traces is used. Second, from the timing information of
 * the individual stations, the direction of the shower is obtained by triangulation. Third, the antenna pattern
 * for this direction is evaluated, and the E-field trace at each station reconstructed from the voltage traces.
 * Finally, the maximum of the envelope of the E-field trace is used as updated timing information for a new
 * iteration of the procedure."; section 5, L83 names keeping
 * the data on the GPU as the remedy for copy-dominated run time). Per event, all on the device:
 *
 *   n_i, w_i = lowest n maximising v0[n]^2 + v1[n]^2 and that maximum          (timing from the voltages)
 *   for it = 0 .. n_iter-1:
 *     (theta, phi) = weighted plane-wave fit of the arrival samples n_i on the flat array `positions`,
 *                    c n_i / fs = c t0 - (u x_i + v y_i), (u, v) = sin(theta) (cos(phi), sin(phi)),
 *                    weights w_i; theta = asin(min(1, |(u,v)|)), phi = atan2(v, u) in [0, 360) degrees;
 *                    no positive weight or a degenerate array gives (0, 0)
 *     unfold every station at (theta, phi) exactly as aera_unfold_batch does (peaks only, except that the
 *     last iteration also writes the E-field traces when efield != NULL)
 *     n_i = peak_idx_i, w_i = peak_amp_i^2
 *
 *   traces    [n_events][n_stations][2][n_samples] real (dtype)   device, 16-byte aligned
 *   positions [n_stations][2] double, metres (x, y)                device
 *   dirs_hist [n_iter][n_events][2] double, degrees                device, out
 *   efield    as in aera_unfold_batch; may be NULL; may alias traces (written in the last iteration only)
 *   amp_hist  [n_iter][n_events][n_stations] real (dtype), idx_hist the same shape int32     device, out
 *   idx0 / w0 [n_events][n_stations] int32 / real (dtype): the voltage timing                 device, out
 *   workspace >= aera_workspace_bytes(AERA_OP_UNFOLD, ...) for n_events. With
 *             aera_workspace_bytes(AERA_OP_RECONSTRUCT, ...) or more (room for the direction-independent band
 *             spectra of every station, 9.7 KB each at configs[1]) the first iteration stores them and the later
 *             ones start from them: no trace re-read, no forward transform (results are bit-identical)
 * Asynchronous on the stream; errors as aera_unfold_batch, plus AERA_ERR_INVALID_ARG for n_iter < 1.
 */
aera_status_t aera_reconstruct_batch(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                                     int n_samples, double fs_hz, const void *traces, const double *positions,
                                     int n_iter, double *dirs_hist, void *efield, void *amp_hist, int32_t *idx_hist,
                                     int32_t *idx0, void *w0, void *workspace, size_t workspace_bytes,
                                     void *cuda_stream);

/* Convergence of the reconstruction loop (section 2: "On convergence, the timing information yields the
 * incident direction of the primary particle"; the paper gives no criterion, reading R21): for every event the
 * first iteration it >= 1 whose fitted direction lies within tol_deg (angle on the unit sphere, degrees) of iteration
 * it - 1, or -1 if none does. The caller runs aera_reconstruct_batch with an upper bound n_iter and reads the direction
 * and peaks of iteration conv_iter[event] (or the last one).
 *   dirs_hist  DEVICE [n_iter][n_events][2] double, as written by aera_reconstruct_batch
 *   conv_iter  DEVICE [n_events] int32, out
 * Asynchronous on the stream. Errors: INVALID_ARG, CUDA. */
aera_status_t aera_reconstruct_convergence(const double *dirs_hist, int n_iter, int n_events, double tol_deg,
                                           int32_t *conv_iter, void *cuda_stream);

/* End-to-end convenience for HOST buffers (the paper's situation: traces live on
 * the host and are copied for every transform).  Same arguments as aera_unfold_batch but every
 * data pointer is a HOST pointer (page-locked memory gives full PCIe speed; pageable works).
 * The batch is cut into event chunks that flow through a 3-stream pipeline
 * (H2D copy | unfold kernels | D2H copy) over device staging buffers owned by the pattern handle
 * (allocated on first use, reused afterwards).  SYNCHRONOUS: results are in the host buffers on
 * return.  efield may be NULL. */
aera_status_t aera_unfold_batch_host(aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                                     int n_samples, double fs_hz, const void *traces_host,
                                     const double *dirs_host, void *efield_host, void *peak_amp_host,
                                     int32_t *peak_idx_host);

/* aera_unfold_batch_host for int16 ADC counts (section 5, L79 and L83: the copies to and from the device, not
 * the transforms, dominate the run time, so the lever of the host path is bytes). The traces cross PCIe as int16 (half
 * the bytes of fp32) and are converted in the kernel exactly as aera_unfold_batch_i16 does; with efield_host == NULL
 * only the peaks come back and no E-field is staged at all. Per station at n_samples = 2048: 8 192 B in + 8 B out
 * (peaks only) or + 16 384 B (E-field), against 16 384 B + 16 392 B of the fp32 call.
 *   traces_host      HOST [n_events][n_stations][2][n_samples] int16 (page-locked memory gives full PCIe speed)
 *   counts_to_volts  HOST [2] double, one factor per channel
 *   efield_host      HOST fp32 [n_events][n_stations][2][n_samples], or NULL (peaks only)
 *   peak_amp_host / peak_idx_host  HOST fp32 / int32 [n_events][n_stations]
 *   pattern          an AERA_F32 pattern
 * SYNCHRONOUS; shares the pattern handle's staging buffers and streams with aera_unfold_batch_host (one call at a time
 * per handle; the buffers grow on demand). Errors as aera_unfold_batch_host and aera_unfold_batch_i16. */
aera_status_t aera_unfold_batch_host_i16(aera_pattern_t *pattern, int n_events, int n_stations, int n_samples, double fs_hz,
                                         const int16_t *traces_host, const double *counts_to_volts, const double *dirs_host,
                                         float *efield_host, float *peak_amp_host, int32_t *peak_idx_host);

/*
 * Batch unfolding without a workspace and without any allocation (the operation of aera_unfold_batch; PAPER.md
 * section 2, L29 steps 3 + 4; section 5: keep the data on the device and the copies out of the loop).
 *
 * For whom: code that is handed its input and output buffers and nothing else. Two cases in practice. (1) A
 * reconstruction module loaded into a host application that owns the device-memory pool: the module may not call
 * cudaMalloc, and often could not if it tried because the pool has taken the whole card. (2) A trigger or
 * monitoring loop with a latency budget: cudaMalloc / cudaFree serialise on a driver lock and synchronise the
 * device, so one allocation anywhere in the loop stalls every stream of the process.
 *
 * The scratch that aera_unfold_batch takes as `workspace` is here an array of AERA_STATIC_SCRATCH_BYTES (32 MiB)
 * built into the library. Every GPU on which the library's code is loaded holds those 32 MiB until the process
 * exits, whether this call is used or not. A batch whose aera_workspace_bytes(AERA_OP_UNFOLD, ...) exceeds the
 * array is refused with AERA_ERR_WORKSPACE (the message gives both numbers); nothing is allocated instead. At
 * BASELINE configs[1] (n_samples = 2048 fp32, fs = 180 MHz) one event needs 20 256 bytes, so up to 1 656 events
 * fit in a call; cut larger batches into several calls.
 *
 * Arguments are those of aera_unfold_batch without workspace / workspace_bytes; results are the same bit for bit
 * (the same kernels run). The call itself makes no cudaMalloc, cudaFree or other allocating call, on the host or
 * on the device. Two things therefore belong to set-up:
 *   - aera_pattern_prepare(pattern, n_samples, fs_hz, stream) once per (pattern, n_samples, fs_hz): it builds the
 *     small plan (twiddle and bin tables) that the other entry points build on first use, which is a cudaMalloc and
 *     a synchronising upload. Without it this call returns AERA_ERR_INVALID_ARG and says so.
 *   - the FIRST call of this entry point on each device looks up the device address of the built-in array (and the
 *     CUDA runtime loads the kernels' code on first launch). Make that first call with that device current, during
 *     set-up, and before any stream capture is begun; later calls on that device do a table look-up only.
 *     Leave aera_profile_enable off (it creates events).
 * All calls on one device share the one array, and it keeps whatever the previous call wrote. Nothing in it needs
 * to start at zero (each call writes every entry it later reads), so consecutive calls on ONE stream are safe as
 * they are. Two calls that can overlap on the GPU -- different streams, or different host threads without ordering
 * between their streams -- race on the array and produce garbage: order them (one stream, or events), or give the
 * second one a workspace of its own through aera_unfold_batch.
 * Errors: as aera_unfold_batch, plus the two above.
 */
#define AERA_STATIC_SCRATCH_BYTES (32u << 20)
aera_status_t aera_unfold_batch_static(const aera_pattern_t *pattern, int dtype, int n_events, int n_stations,
                                       int n_samples, double fs_hz, const void *traces, const double *dirs,
                                       void *efield, void *peak_amp, int32_t *peak_idx, void *cuda_stream);

/* Set-up for aera_unfold_batch_static (useful before any entry point when the first hot call must not allocate or
 * synchronise): builds and caches the plan of (n_samples, fs_hz) in the pattern handle. Allocates device memory and
 * synchronises the stream once; a second call for the same pair is a no-op. Errors: INVALID_ARG, UNSUPPORTED_N, BAND,
 * ALLOC, CUDA. */
aera_status_t aera_pattern_prepare(aera_pattern_t *pattern, int n_samples, double fs_hz, void *cuda_stream);

/* AERA_STATIC_SCRATCH_BYTES as the loaded library was built (for bindings that cannot read the macro). */
size_t aera_static_scratch_bytes(void);

/* Kernel selection, for tests and tuning. 0 = automatic (specialised kernels where available),
 * 1 = always the generic radix-2 kernel. Process-wide. Returns the previous value. */
int aera_set_kernel_variant(int variant);

/* Opt-in for the long-trace kernel (fp32, n_samples = 65536): its inter-pass scratch (about 70 MB in the workspace) is
 * meant to live in the L2, and its lines carry an evict_last hint that only holds inside the persisting carve-out of
 * the L2. That carve-out (cudaLimitPersistingL2CacheSize) is device-wide state shared with everything else the process
 * runs, so the library leaves it alone by default (megabytes < 0). With megabytes >= 0 the next long-trace launch on
 * each device sets the limit to min(megabytes, device maximum) MB (pass a large number for the maximum, 79 MB on the
 * B200; 0 switches the carve-out off) and it stays so until changed. Measured on configs[4]: DRAM traffic per station
 * 1.11 MB with the maximum against 1.83 MB without (1.05 MB algorithmic); throughput within 3 % either way, because
 * that kernel is not DRAM-bound. Process-wide. Returns the previous request. */
int aera_set_long_trace_l2_persist(int megabytes);

/* Number of kernel launches this library has enqueued since load (monotonic, all threads). */
unsigned long long aera_launch_count(void);

/* Per-kernel device timing with CUDA events recorded on the stream each kernel is launched on
 * (used by bench.py for the roofline figures; off by default, costs two event records per launch).
 * aera_profile_enable(1) clears earlier records and starts recording; (0) stops. Returns the
 * previous state. aera_profile_read waits for the recorded events of one kernel and returns the
 * summed duration and the number of launches. kernel_id: 0 table repack, 1 pattern
 * evaluation + 2x2 inverse (per event/direction), 2 batched unfold, 3 scan forward, 4 scan inverse. */
int aera_profile_enable(int on);
aera_status_t aera_profile_read(int kernel_id, double *total_ms, long *launches);

/* Measured ALU throughput of the current device: the denominator of the "alu" roofline that bench.py reports for
 * the FP32-pipe-bound direction scan (BASELINE north_star: "FP32/FP64 pipe utilisation for the scan mode"), in
 * place of a number derived from unit counts and clocks. A register-only chain of independent fused multiply-adds
 * on every SM (warps_per_sm warps each, 1..32) is timed with CUDA events (best of 3).
 *   kind 0: packed fp32 (fma.rn.f32x2, the warp kernels' instruction), 1: scalar fp32, 2: fp64
 *   lane_fma_per_s  out: fused multiply-adds per second over the whole device (x 2 = FLOP/s)
 *   sm_count, sm_clock_khz  out: cudaDevAttrMultiProcessorCount, cudaDevAttrClockRate (may be NULL). The latter is the
 *                           device's MAXIMUM SM clock, not the clock during the measurement: a per-clock figure derived
 *                           from it understates the pipe when the device throttles (bench.py --peaks also reports one on
 *                           the clock nvidia-smi observed)
 * SYNCHRONOUS (default stream); allocates and frees a small device buffer. Errors: INVALID_ARG, ALLOC/CUDA. */
aera_status_t aera_measure_alu_peak(int kind, int warps_per_sm, double *lane_fma_per_s, int *sm_count, int *sm_clock_khz);

/* Which kernel family the most recent aera_unfold_batch / aera_fold_batch / aera_scan_directions /
 * aera_reconstruct_batch call of this thread dispatched to: a static string, one of "unfold_w32" (fp32 N = 2048),
 * "unfold_t1k_f32|f64" (N = 1024), "unfold_t2k_f64" (N = 2048), "unfold_t4k_f32|f64" (N = 4096), "unfold_t8k_f32|f64"
 * (N = 8192), "unfold_t16k_f32" (N = 16384), "unfold_long_f32" (fp32 N = 65536, band below N/4), "scan_w32" (fp32
 * N = 2048 scan), "generic" (every other size, and up-sampling); "" before the first call. Lets a caller see that a
 * size fell to the slower generic radix-8 kernels. */
const char *aera_last_kernel(void);

/* Message for the most recent non-OK status on this thread ("" if none). Static storage. */
const char *aera_last_error(void);

/* Library version string, e.g. "aera_unfold 0.1 (sm_100a)". */
const char *aera_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AERA_UNFOLD_H */

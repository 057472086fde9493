/* tdlike.h - C ABI of the B200-native time-domain Gaussian log-likelihood library.
 *
 * The operation (arxiv 2603.06010; line numbers are /root/reference/PAPER.md):
 *   C_s[i][j] = rho_s(|i-j|)                       symmetric Toeplitz noise covariance   (Eq. 5,  :107)
 *   <x, y>_s  = x^T C_s^{-1} y                      time-domain inner product             (Eq. 6,  :113)
 *   lnL       = const - 1/2 <d - h, d - h>          exact Gaussian likelihood             (Eq. 7,  :125; Eq. 10, :142)
 *   segments / detectors are independent blocks whose log-likelihoods are summed        (items 1-3, :148-162)
 *   <.,.> is evaluated exactly through the Gohberg-Semencul formula                      (Eq. 14, :241-246)
 *       C^{-1} = (1/x_1)(L_x L_x^T - R_x^T R_x),  C x = e_1,
 *   each triangular-Toeplitz product by circulant embedding + FFT, m >= 2n-1           (Eqs. 15-16, :246-252)
 *   or, for short segments, as a dense Toeplitz-by-matrix contraction (the GEMV of :219-227, batched).
 *
 * All entry points return a td_status and never abort or throw.  Nothing here allocates or
 * frees caller memory.  There is no CPU fallback: every call needs a CUDA device.
 *
 * Threads and streams.  A handle must not be used from two host threads at once.  The handle owns device scratch
 * (the workspace of the long-segment kernels, z and u = C^{-1} d of the data vector for td_inner_batch, the synthesis
 * panel of td_loglike_family_batch): calls issued on ONE stream are ordered by the stream; a call issued on a
 * DIFFERENT stream than the previous scratch-using call first waits (cudaStreamWaitEvent) for that call, so one thread
 * alternating between streams gets correct, serialised results.  Inside a CUDA stream capture the library records and
 * waits on nothing: the captured graph's own dependencies order the work, and the caller must not replay such a graph
 * concurrently with other calls on the same handle.
 *
 * Allocation.  td_create allocates everything whose size does not depend on the batch, sets every kernel attribute and
 * caches every occupancy figure.  The device-pointer calls (td_loglike_batch, td_inner_batch) never allocate or
 * synchronise: they only enqueue kernels, and can be captured into a CUDA graph.  Buffers that grow with the batch
 * (host staging, the synthesis panel) are sized by td_reserve, or on first use when the caller did not reserve.
 */
#ifndef TDLIKE_H_
#define TDLIKE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct td_handle td_handle; /* opaque; owns device-side generators, spectra, workspace */

typedef enum {
  TD_OK = 0,
  TD_EINVAL = 1,       /* bad argument (null pointer, non-positive length, ldh < N_tot, ...) */
  TD_ENOTSPD = 2,      /* an ACF is not symmetric-positive-definite (or not finite)           */
  TD_ENOMEM = 3,       /* host or device allocation failed                                    */
  TD_ECUDA = 4,        /* a CUDA runtime call / kernel launch failed                          */
  TD_EUNSUPPORTED = 5  /* valid request this build cannot serve (e.g. forced path too large)  */
} td_status;

/* td_path: evaluation path selector for td_set_path / reported by td_get_info.
 * TD_PATH_AUTO: per size class (power-of-two padded length), the dense kernels for short segments, the FFT kernels
 * otherwise; all accumulate into the same outputs within one call.  Measured crossovers:
 * td_loglike_batch - classes whose segments are all <= 512 samples: CDO contraction (segments under 65 samples: the
 * Gohberg-Semencul dense kernel); td_inner_batch - classes whose segments are all <= 512 samples: Gohberg-Semencul. */
enum { TD_PATH_AUTO = 0, TD_PATH_FFT = 1, TD_PATH_DENSE = 2,
       TD_PATH_DOT = 3, /* reported by td_get_info only: <d,h_b> evaluated as u . h_b, u = C^{-1} d */
       TD_PATH_CDO = 4  /* td_loglike_batch as the batched triangular contraction Y = L^{-1} X with the cached whitening
                           operator (the paper's "CDO" route) for EVERY segment (AUTO uses it for
                           classes up to 512 samples, profiles/r02_cdo.md, r02_short_segments.md); segments up to 1024 samples; the first
                           td_set_path(TD_PATH_CDO) builds the L^{-1} that td_create has not (8 N^2 bytes per
                           segment); td_inner_batch keeps using the dense path */ };

/* td_create - one-time setup (PAPER.md:215 "done once ... cached"; :241-246 Eq. 14 generator).
 *   acf          HOST pointer, sum_s seg_lengths[s] doubles: per-segment autocorrelation
 *                functions concatenated; segment s holds rho_s(0..N_s-1) (Eq. 11, :148-154:
 *                a segment of N_s samples uses lags 0..N_s-1), rho_s(0) > 0.
 *   seg_lengths  HOST pointer, n_seg entries, each >= 1.
 *   n_seg        number of disjoint segments / detectors (>= 1).
 *   device       CUDA device ordinal that will own the handle.
 *   out          receives the handle on success; untouched on failure.
 * Per segment it runs a Levinson-Durbin recursion on the device, giving the prediction-error
 * filter a (a_0 = 1) and variance v with C a = v e_1 (so x = a/v, x_1 = 1/v in Eq. 14),
 * b = (0, a_{N-1}, ..., a_1), the pre-transformed generator spectra for the FFT path and
 * log det C_s as a by-product.  Synchronous (returns after the device work completed).
 * Errors: TD_EINVAL, TD_ENOTSPD (recursion met E_k <= 0 or a non-finite value), TD_ENOMEM, TD_ECUDA.
 */
td_status td_create(const double* acf, const int64_t* seg_lengths, int n_seg, int device,
                    td_handle** out);

/* td_destroy - frees everything the handle owns.  NULL is accepted. */
td_status td_destroy(td_handle* h);

/* td_loglike_batch - the hot path (Eq. 10 summed over segments, :142, :162).
 *   d    DEVICE pointer, N_tot doubles: kept samples only, segments concatenated in order
 *        (gap samples are not passed; Eq. 12 read as independent blocks, reading A5).
 *   H    DEVICE pointer, row-major [B][ldh] doubles, ldh >= N_tot; row b = template h_b with
 *        the same segment packing as d.
 *   ldh  leading dimension of H in elements.
 *   B    number of templates; B == 0 is a no-op returning TD_OK.
 *   out  DEVICE pointer, B doubles: out[b] = -1/2 sum_s (d_s - h_bs)^T C_s^{-1} (d_s - h_bs)
 *        (the additive constant of Eq. 7 is NOT included; see td_get_info for log det).
 *   stream  a cudaStream_t (as void*; NULL = legacy default stream).
 * Asynchronous: kernels are enqueued on `stream`; no host synchronisation, no allocation (CUDA-graph capturable).
 * The residual d - h_b and the filtered vectors are never written to HBM on the fused path.
 * NaN/Inf in row b of H (or in d) propagate to out[b].
 */
td_status td_loglike_batch(td_handle* h, const double* d, const double* H, int64_t ldh,
                           int64_t B, double* out, void* stream);

/* td_inner_batch - cross terms of Eq. 13 (:177-181): out_dh[b] = <d, h_b>, out_hh[b] = <h_b, h_b>,
 * both summed over segments.  Either output may be NULL (not computed / not written).
 * Same layouts, ownership and stream semantics as td_loglike_batch.
 * Identity: -2 * loglike[b] = <d,d> - 2 <d,h_b> + <h_b,h_b>;  <d,d> is td_inner_batch with H = d, B = 1.
 * With out_hh == NULL under TD_PATH_AUTO (segments up to 16384 samples) the cross term is evaluated as the batched dot
 * product u . h_b against u = C^{-1} d, computed once per call from the Gohberg-Semencul form (the paper's cached
 * whitened data, :225, :306, taken one step further): one pass over H, HBM-bound; td_get_info then reports TD_PATH_DOT.
 */
td_status td_inner_batch(td_handle* h, const double* d, const double* H, int64_t ldh,
                         int64_t B, double* out_dh, double* out_hh, void* stream);

/* td_loglike_batch_host - td_loglike_batch for HOST buffers (the end-to-end call).
 *   d, H, out are HOST pointers with the layouts above (H ideally page-locked, otherwise the
 *   copies are not asynchronous).  The library copies d once, streams H to the device in row
 *   chunks through two staging buffers on an internal copy stream so that the host-to-device
 *   copy of chunk k+1 overlaps the kernels of chunk k, and copies out back.
 * SYNCHRONOUS: returns after out[] is complete.  `stream` is the compute stream (NULL = default).
 */
td_status td_loglike_batch_host(td_handle* h, const double* d, const double* H, int64_t ldh,
                                int64_t B, double* out, void* stream);

/* td_family: analytic template families of td_loglike_family_batch (rows of 5 parameters; t_i = i / fs counted from the
 * segment's first sample, n = the segment's length):
 *   TD_FAMILY_RINGDOWN      (A, f, tau, phi, t0):      A exp(-(t_i - t0)/tau) cos(2 pi f (t_i - t0) + phi) for t_i >= t0, else 0
 *   TD_FAMILY_SINE_GAUSSIAN (A, f, w, phi, t0):        A exp(-((t_i - t0)/w)^2) cos(2 pi f t_i + phi)
 *   TD_FAMILY_CHIRP         (A, f0, fdot, phi, alpha): A tukey_alpha(i / (n - 1)) cos(2 pi (f0 t_i + fdot t_i^2 / 2) + phi)
 * (the template families of BASELINE.json's configs c1/c2/c5, c3 and c4). */
enum { TD_FAMILY_RINGDOWN = 0, TD_FAMILY_SINE_GAUSSIAN = 1, TD_FAMILY_CHIRP = 2 };

/* td_loglike_family_batch - td_loglike_batch for templates given by PARAMETERS (waveform
 * generation and placement, moved onto the device for the analytic families of the configs):
 *   family  one of td_family.
 *   params  DEVICE pointer, row-major [B][n_seg][5] doubles, one row per (template, segment / detector), in the
 *           segment's own time.  A detector projection F+ h_c + Fx h_s of a ringdown with a time shift dt (:164, :209)
 *           is such a row: amplitude A hypot(F+, Fx), phase phi - atan2(Fx, F+), onset t0 + dt; a segment that starts at
 *           time ts of a longer record takes t0 - ts (and phi + 2 pi f ts for the sine-Gaussian).
 *   fs      sampling rate in Hz (> 0);  d, out, stream as in td_loglike_batch.
 * The rows are synthesised into a scratch panel owned by the handle, chunk by chunk (about 128 MB; td_reserve sizes it),
 * and each chunk goes through the same kernels as td_loglike_batch; small ringdown batches (up to 2 x the SM count, segments
 * of 513..4096 samples) are synthesised inside the first pass of the fused kernel instead: one launch, no panel
 * (profiles/r02_ring_fused.md has both routes measured).  Asynchronous on `stream`.
 * Errors: TD_EINVAL (unknown family, fs <= 0, null pointers), TD_ENOMEM, TD_ECUDA. */
td_status td_loglike_family_batch(td_handle* h, const double* d, int family, const double* params, int64_t B, double fs,
                                  double* out, void* stream);

/* td_loglike_family_batch_host - the same from HOST buffers (d, params, out): 40 bytes per template and segment cross
 * the bus instead of 8 N_s.  SYNCHRONOUS: returns after out[] is complete. */
td_status td_loglike_family_batch_host(td_handle* h, const double* d, int family, const double* params, int64_t B,
                                       double fs, double* out, void* stream);

/* td_reserve - sizes every batch-dependent buffer of the handle for calls of up to B_max templates: the partial sums of
 * the long-segment kernels, the device staging of td_loglike_batch_host (H chunks, d, out), the synthesis panel and the
 * parameter buffer of td_loglike_family_batch(_host).  After it, no entry point allocates for B <= B_max (so the
 * parameter entry point, too, is allocation-free and capturable).  Grow-only; synchronous (cudaMalloc).
 * Errors: TD_EINVAL (B_max < 0), TD_ENOMEM, TD_ECUDA. */
td_status td_reserve(td_handle* h, int64_t B_max);

/* td_set_path - force the evaluation path for subsequent calls (TD_PATH_AUTO restores the
 * chooser).  TD_PATH_DENSE / TD_PATH_CDO on a handle with a segment longer than the dense paths support
 * (1024 samples) return TD_EUNSUPPORTED and leave the setting unchanged. */
td_status td_set_path(td_handle* h, int path);

/* td_set_fft_variant - which implementation serves the FFT path: 0 = automatic (fused
 * shared-memory kernel where a segment's transform fits one SM; 2-CTA cluster kernel for 4097..8192 samples; segments of
 * 8193..65536 samples on the group kernel, td_group16.cuh: one cooperative launch, 4 / 8 / 16 CTAs per template exchanging
 * the two cross passes through L2, when the device can co-host such a group; staged global-memory kernels
 * otherwise; ringdown parameter rows synthesised inside the fused kernel's first pass), 1 = as 0 but
 * td_loglike_family_batch always synthesises into the scratch panel first (the r01 route; tests, profiling),
 * 2 = force the staged kernels for every segment (tests, profiling), 3 = as 0 but segments of 32769..65536 samples run on
 * the 16-CTA cluster kernel (td_cluster16.cuh: the 3 MB of spectra of one template in distributed shared memory; measured
 * slower than the staged kernels on B200, profiles/r02_c4_cluster16.md; TD_EUNSUPPORTED when the handle has no such
 * segment or the device cannot host a 16-CTA cluster), 4 = the explicit name of what 0 does for segments of 8193..65536
 * samples (TD_EUNSUPPORTED when the handle has no such segment or the device cannot co-host a group). */
td_status td_set_fft_variant(td_handle* h, int variant);

/* td_precision: arithmetic of the FFT-path evaluation (td_set_precision). */
enum { TD_PREC_F64 = 0, TD_PREC_F32 = 1 };

/* td_set_precision - FP32 evaluation with FP64 setup (III.C.3: "it is possible to carry out all the
 * analysis with FP32 with appropriate normalization.  However, the necessary matrices and whitening operators should be
 * precomputed in FP64"; :268).  TD_PREC_F32: the Levinson-Durbin recursion, the generator spectra and the twiddles stay
 * fp64 (td_create) and are rounded once; per template the residual d - h is formed in fp64 from the fp64 inputs, divided
 * by sqrt(rho_s(0)) (the normalisation; the spectra carry the inverse factor) and rounded once; S2-S4 (both FFTs, the
 * generator product) run in fp32; the sums of squares are fp32 per thread and fp64 across threads, segments and in out[].
 * The interface (double d, H, out) is unchanged.  Serves segments of 513 samples and more (fp32 builds of the fused, cluster
 * and staged kernels); shorter segments (the dense paths) and the dot-product cross term keep evaluating in fp64.
 * Accuracy: |out - exact| <= 2e-5 * max(|exact|, 1) per template (DESIGN.md 6.7 derives it; observed ~1e-6); the fp64
 * default keeps the 1e-9 bar.  The first call builds the fp32 tables (synchronous, allocates); later calls only switch.
 * Errors: TD_EINVAL (unknown precision), TD_EUNSUPPORTED (no segment of the handle has an fp32 kernel; the setting is
 * unchanged), TD_ENOMEM, TD_ECUDA. */
td_status td_set_precision(td_handle* h, int precision);

/* td_get_info - queries.  Any output pointer may be NULL.
 *   n_tot      sum of segment lengths
 *   n_seg      number of segments
 *   v          HOST array [n_seg]: prediction-error variance v_s = 1/(C_s^{-1})_{00}
 *   logdet     HOST array [n_seg]: log det C_s = sum_k log E_k
 *   last_path  path actually used by the last batch call (0 if none yet): TD_PATH_CDO / TD_PATH_DENSE if every segment went
 *              through the dense kernels (CDO if the cached-L^-1 contraction took part), TD_PATH_DOT for the dot-product
 *              cross term, TD_PATH_FFT otherwise
 */
td_status td_get_info(const td_handle* h, int64_t* n_tot, int* n_seg, double* v, double* logdet,
                      int* last_path);

/* td_get_generator - copies segment s's prediction-error filter a (N_s doubles, a[0] = 1) to the
 * HOST buffer `a`.  For tests of the setup kernel (C a = v e_1). */
td_status td_get_generator(const td_handle* h, int seg, double* a);

/* td_last_launches - number of kernels of this library launched by the last batch call on
 * this handle (evidence for bench.py's gpu_launches). */
int td_last_launches(const td_handle* h);

/* td_strerror - static string for a status code. */
const char* td_strerror(td_status s);

/* ---- allocation-free evaluation ------------------------------------------------------------------------------------
 * For callers that cannot allocate device memory at call time (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc).  td_loglike_batch_static computes what td_loglike_batch computes (Eq. 10,
 * PAPER.md:142; FFT route of Eqs. 14-16, :241-252) with the staged kernels (forward passes - untangle x generator - inverse
 * passes - fused reduction on a global-memory workspace), whose workspace is NOT the handle's cudaMalloc'ed buffers but a
 * file-scope device array of TD_STATIC_SCRATCH_BYTES inside the library image.  The call itself - and td_static_setup -
 * call no cudaMalloc / cudaFree / allocating library routine; the handle (td_create) must exist beforehand.
 *
 * Limits and ownership:
 *  - every GPU that loads this library holds TD_STATIC_SCRATCH_BYTES (16 MiB) of device memory for the array until the
 *    process exits, whether or not the entry point is used;
 *  - one template of a size class (segments padded to M = 2^k samples) needs 48 M + 16 ceil(M / (128 r)) bytes of it
 *    (r = 2..16 the first radix): segments of at most 262144 samples.  A handle with a longer segment is refused with
 *    TD_EUNSUPPORTED before anything is launched (td_static_last_error says how many bytes were needed); B is unlimited
 *    (templates run in chunks of as many as the array holds);
 *  - ONE array per GPU, shared by every handle, thread and stream of the process: two calls that overlap on the GPU
 *    (different streams, or graphs replayed concurrently) race on it and return garbage; serialise them.  The array keeps the
 *    last call's contents; nothing in it has to start at zero (every element a call reads it has written before), so
 *    nothing is cleared;
 *  - always fp64 and always the staged kernels, whatever td_set_path / td_set_fft_variant / td_set_precision say: it is
 *    slower than td_loglike_batch wherever that runs a fused kernel.  Results agree with td_loglike_batch to rounding
 *    (1e-9 relative, the parity tolerance; tests/test_zz_no_alloc.py).
 * Arguments, layout, stream semantics and errors otherwise as td_loglike_batch: d, H, out DEVICE pointers. */
#define TD_STATIC_SCRATCH_BYTES (16u << 20)
td_status td_loglike_batch_static(td_handle* h, const double* d, const double* H, int64_t ldh,
                                  int64_t B, double* out, void* stream /* cudaStream_t */);

/* td_static_setup - resolves the device address of the array on `device` (cudaGetSymbolAddress, once per device) and
 * configures the two shared-memory kernels of the staged pipeline there.  Optional: the first td_loglike_batch_static on a
 * device does the same; call it beforehand when that first call would be inside a stream capture.  TD_ECUDA on failure. */
td_status td_static_setup(int device);

/* td_static_scratch_bytes - TD_STATIC_SCRATCH_BYTES of the loaded library.
 * td_static_last_error - what the last td_static_setup / td_loglike_batch_static of the calling thread refused, in words
 * ("" after a success); static storage, valid until the thread's next such call. */
size_t td_static_scratch_bytes(void);
const char* td_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TDLIKE_H_ */

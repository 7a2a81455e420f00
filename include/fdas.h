/*
 * fdas.h -- C ABI of libfdas.so: the Fourier Domain Acceleration Search hot path of
 * arXiv 1511.07343 (Dimoudi & Armour) as hand-written CUDA for NVIDIA B200 (sm_100a).
 *
 * Citations are "PAPER.md:<line>" (the paper text) and "BJ:..." (BASELINE.json).
 *
 * The path (the seven steps of section 4; Eq. (1)):
 *   series --fdas_spectrum--> normalised complex spectrum
 *          --fdas_correlate-> f-fdot power plane (and/or fused candidates)
 *          --fdas_harmsum / fdas_candidates--> candidate list
 * with the template bank built once by fdas_build_templates.
 *
 * Conventions
 *   - "d_" pointers are DEVICE pointers, "h_" pointers are HOST pointers. All device
 *     buffers are caller-owned (allocate them with PyTorch or cudaMalloc); the library
 *     never allocates in the d_* hot calls. The plan owns only the template bank and a
 *     few KB of metadata; fdas_search_host additionally owns a scratch arena it
 *     allocates on first use.
 *   - Alignment of device pointers (FDAS_E_INVALID otherwise; what cudaMalloc and PyTorch return
 *     always qualifies): d_series and d_spectrum 8 bytes, d_plane 16 bytes for fdas_correlate and
 *     4 bytes for fdas_harmsum / fdas_candidates, candidate lists and counters 4 bytes, the
 *     workspace 256 bytes.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream). Every d_* hot
 *     call only enqueues work and returns; nothing synchronises.
 *   - Return value: FDAS_OK (0) or a negative FDAS_E_* code. No exceptions, no exit().
 *   - Notation: N = n_samples (power of two); n_bins = N/2 (Fourier bins 1..N/2 are kept,
 *     plane column c <-> bin bin0 + c, bin0 = 1); m = template_width; L = segment_len;
 *     n_z = 2*z_max/dz + 1, z_i = -z_max + i*dz; nset = 1 + interbin;
 *     n_templates = n_z*nset (template t = zi*nset + s); n_cols = n_bins*nset;
 *     step = L - m outputs kept per overlap-save segment; n_seg = ceil(n_bins/step).
 */
#ifndef FDAS_H
#define FDAS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define FDAS_OK            0
#define FDAS_E_INVALID    -1   /* bad argument (see each call) */
#define FDAS_E_STATE      -2   /* templates not built / option set after build */
#define FDAS_E_WORKSPACE  -3   /* workspace missing or misaligned */
#define FDAS_E_CUDA       -4   /* a CUDA call failed; fdas_strerror(code) gives the sticky text */
#define FDAS_E_NOMEM      -5   /* host or device allocation failed (plan create / host API only) */

/* fdas_plan_set_option keys */
#define FDAS_OPT_INTERBIN     1  /* 0/1: add the half-bin template set (BJ:configs[1]); default 0 */
#define FDAS_OPT_MAX_BATCH    2  /* largest n_batch the calls will see (sizes workspace_bytes); default 1 */
#define FDAS_OPT_QUAD_POINTS  3  /* quadrature points of the template generator; default 32768 */
/* Tuning keys: launch geometry / instruction selection only, results do not depend on them; may be set at
 * any time; 0 = the default.  Kept for A/B timing (bench.py --ab). */
#define FDAS_OPT_TUNE_SCALAR     101  /* 1: scalar FFMA butterflies in the L = 2048 segment kernel (default: packed FFMA2) */
#define FDAS_OPT_TUNE_T_CHUNKS   102  /* template chunks per segment in the L = 2048 segment kernel (default ceil(n_t/29)) */
#define FDAS_OPT_TUNE_HS_SECTORS 103  /* angular sectors of the harmonic-sum tile order, 1..64 (default 16) */
#define FDAS_OPT_TUNE_HS_ROWS    104  /* warps per CTA of the harmonic-sum kernel, 1..8 (default 4) */
#define FDAS_OPT_TUNE_HS_VARIANT 105  /* 1: 128-column harmonic-sum tiles (default 64) */
#define FDAS_OPT_TUNE_STAGE_TEMPLATES 107 /* 1: L = 2048 segment kernel with four segments per CTA that share every
                                          * template spectrum through shared memory (one 16 KB bulk copy per CTA and
                                          * template instead of one L2 read per segment); default 0 until it is timed */
#define FDAS_OPT_TUNE_SPEC_SELFTEST 108 /* before build: 0 = fdas_build_templates checks the TMA-staged spectrum passes against
                                        * the generic kernels on one seeded series (default), 1 = skip, 2 = test hook:
                                        * behave as if the check had failed */
#define FDAS_OPT_TUNE_SPEC_GENERIC 106 /* 1: the generic two-pass spectrum kernels at every length (default: the
                                        * TMA-staged multi-pass transform from 2^13 samples on) */

typedef struct fdas_plan fdas_plan;

/* One candidate, 12 bytes.  col = plane column; Fourier frequency r = bin0 + col/nset;
 * z = -z_max + zi*dz; nharm = number of harmonics summed (1 for fdas_correlate and
 * fdas_candidates); power = (summed) normalised power. */
typedef struct {
    int32_t col;
    int16_t zi;
    int16_t nharm;
    float   power;
} fdas_cand;

typedef struct {
    int64_t n_samples, n_bins, n_cols;
    int32_t bin0, n_z, n_templates, width, seg_len, step, n_seg, interbin;
    double  z_max, dz;
    size_t  workspace_bytes;   /* size of d_workspace for fdas_spectrum at MAX_BATCH */
} fdas_info;

/* Select the CUDA device the calling thread's subsequent fdas_* calls use (the library
 * links its own CUDA runtime; call this with the same index PyTorch uses). */
int fdas_set_device(int32_t device);

/* Create a plan for series of n_samples real samples searched with templates
 * z = -z_max .. z_max step dz ("multiple templates"; z = fdot*T^2 = bins
 * drifted over the span), each an FIR of `template_width` taps, by
 * overlap-save with segments of `segment_len` bins (PAPER.md:49 step 3).
 * FDAS_E_INVALID unless: n_samples a power of two with 2*segment_len <= n_samples <= 2^25 (the fp32 twiddle
 * arguments k/N are exact up to there);
 * segment_len in {256, 512, 1024, 2048, 4096}; template_width even, >= 2 and
 * <= segment_len/2; dz > 0, z_max >= 0 and z_max/dz an integer; n_z <= 32767. */
int fdas_plan_create(fdas_plan** out, int64_t n_samples, double z_max, double dz,
                     int32_t template_width, int32_t segment_len);

/* Options 1..3 must be set before fdas_build_templates (else FDAS_E_STATE); tuning keys any time. */
int fdas_plan_set_option(fdas_plan* plan, int32_t key, int64_t value);

int fdas_plan_info(const fdas_plan* plan, fdas_info* out);

/* Initialisation stage ("computation of the templates"): for every z and
 * tap j the conjugate ("the complex conjugate of the filter") of the
 * Fourier response of a unit-amplitude constant-fdot chirp,
 *   T_z[j] = conj R_z(d_j),  R_z(d) = int_0^1 exp(2 pi i [(-d - z/2) u + (z/2) u^2]) du,
 *   d_j = j - m/2 (+1/2 for the interbin set),
 * evaluated in fp64 on the device, stored fp32; then the length-L spectrum of the
 * index-reversed, zero-padded taps with the 1/L of the inverse FFT folded in
 * (PAPER.md:49 step 5 "complex multiply - scale").  Allocates the bank (device memory
 * owned by the plan), enqueues on `stream`, and synchronises that stream once. */
int fdas_build_templates(fdas_plan* plan, void* stream);

/* Device status word of the plan, *out = 0 if all is well.  Bit 0 (FDAS_STATUS_COPY_TIMEOUT): a kernel gave up
 * waiting for an asynchronous (TMA) copy -- its waits are bounded so that a mistake shows up here and not as
 * a hung GPU; the results of that call are then undefined.  Synchronous (a 4-byte device-to-host copy): call it
 * after synchronising the stream, not in the hot loop. */
#define FDAS_STATUS_COPY_TIMEOUT 1u
#define FDAS_STATUS_TMA_FALLBACK 2u   /* the init-stage comparison of the TMA-staged spectrum passes with the generic
                                       * kernels failed: the plan uses the generic kernels (slower, correct) */
int fdas_plan_status(const fdas_plan* plan, uint32_t* out);

/* Test hook: copy the fp32 taps to host, h_re_im[(t*m + j)*2 + {0,1}] = {Re, Im} T_t[j].
 * Synchronous. FDAS_E_STATE before build. */
int fdas_get_templates(const fdas_plan* plan, float* h_re_im);

/* PAPER.md:49 step 2 ("Real to complex DFT of the time series") + normalisation
 * (BJ:configs[0] "keep bins 1..N/2, normalise by sqrt(mean |F_k|^2)").
 *   d_series   float[n_batch][N]            in
 *   d_spectrum float2[n_batch][n_bins]      out: S[c] = F_{c+1}/sqrt(mu)   (interleaved re,im)
 *   d_meanpow  float[n_batch]               out: mu = mean_{k=1..N/2} |F_k|^2 (may be NULL)
 *   d_workspace  >= info.workspace_bytes, 256-byte aligned (FDAS_E_WORKSPACE otherwise)
 * F_k = sum_n x_n exp(-2 pi i k n / N) (forward sign -, unnormalised). */
int fdas_spectrum(fdas_plan* plan, const float* d_series, int32_t n_batch,
                  float* d_spectrum, float* d_meanpow, void* d_workspace, void* stream);

/* PAPER.md:49 steps 3-7 fused in one kernel: overlap-save window -> forward FFT ->
 * multiply by every template spectrum -> inverse FFT -> |.|^2 -> discard edges ->
 * plane and/or candidates.  Computes Eq. (1) for every z and bin:
 *   P[b][zi][c*nset + s] = | sum_j S[c + j - m/2 + s] T_{zi,s}[j] |^2 , S = 0 outside [0, n_bins).
 *   d_spectrum float2[n_batch][n_bins]        in
 *   d_plane    float[n_batch][n_z][n_cols]    out, or NULL (fused mode: the plane is not stored)
 *   threshold, d_cands[n_batch][capacity], d_counts[n_batch]: if d_cands != NULL, every
 *       cell with P > threshold (strict) is appended to its batch entry's list (nharm = 1).
 *       The call zeroes d_counts first; d_counts[b] receives the TRUE number found, records
 *       beyond `capacity` are dropped (overflow is not an error; compare count to capacity).
 *       Record order is unspecified.
 *   d_workspace: unused by this call (may be NULL).
 * FDAS_E_INVALID if both d_plane and d_cands are NULL. */
int fdas_correlate(fdas_plan* plan, const float* d_spectrum, int32_t n_batch,
                   float* d_plane, float threshold, fdas_cand* d_cands, uint32_t* d_counts,
                   uint32_t capacity, void* d_workspace, void* stream);

/* Incoherent harmonic summing (BJ:configs[4]; "pulse harmonics") of ONE
 * integer-bin plane float[n_z][n_bins] (FDAS_E_INVALID on an interbinned plan, or if the plane has
 * 2^31 cells or more), for
 * H in {1,2,4,..,max_harm}, max_harm in {1,2,4,8,16}:
 *   k = bin0 + col, zeta = zi - (n_z-1)/2,
 *   k_h = floor((k h + H/2)/H), zeta_h = sgn(zeta) floor((|zeta| h + H/2)/H),
 *   S_H(k, zeta) = sum_{h=1..H} P[zeta_h][k_h - bin0]   (terms with k_h < bin0 are 0).
 * Appends (col, zi, nharm = H, power = S_H) for every cell and stage with
 * S_H > h_thresholds[log2 H] (strict).  h_thresholds: HOST array of log2(max_harm)+1 floats.
 * d_count: one uint32, zeroed by the call, receives the true count (overflow as above). */
int fdas_harmsum(fdas_plan* plan, const float* d_plane, int32_t max_harm,
                 const float* h_thresholds, fdas_cand* d_cands, uint32_t* d_count,
                 uint32_t capacity, void* stream);

/* Threshold + compaction over ONE existing plane float[n_z][n_cols]: every cell with
 * P > threshold (strict) -> (col, zi, 1, P).  d_count as in fdas_harmsum. */
int fdas_candidates(fdas_plan* plan, const float* d_plane, float threshold,
                    fdas_cand* d_cands, uint32_t* d_count, uint32_t capacity, void* stream);

/* Time-domain acceleration trial ("resampling the time series according to a time offset
 * caused by the constant acceleration, followed by a standard periodicity search"): with u = n/N the
 * offset, referred to mid-span, is beta (u^2 - u), so beta = z/(2 r0) turns a signal of mean frequency r0
 * drifting z bins into a tone at r0.  d_out[m] = d_series[min(N-1, floor(u N + 1/2))] with u the root
 *   u = 2u' / [(1 - beta) + sqrt((1 - beta)^2 + 4 beta u')],  u' = m/N,   of  u + beta (u^2 - u) = u',
 * the index being decided in fp64 with separately rounded operations.  d_series, d_out: float[N], distinct
 * buffers, d_out 16-byte aligned; |beta| < 1/2 (FDAS_E_INVALID otherwise).  The periodicity search of d_out is
 * fdas_spectrum followed by fdas_correlate / fdas_candidates on a plan with z_max = 0 (its single template
 * is the delta, so the plane is |S|^2). */
int fdas_resample(fdas_plan* plan, const float* d_series, double beta, float* d_out, void* stream);

/* Host-buffer convenience path (what bench.py's "e2e" times): for each of n_batch series in
 * HOST memory, copy to the device, run spectrum -> correlate -> harmonic sum, and copy the
 * candidate list back.  max_harm = 0 selects the fused threshold mode of fdas_correlate
 * (plane not stored, h_thresholds[0] is the threshold); otherwise the plane is stored in
 * scratch and fdas_harmsum runs on it.  h_cands[n_batch][capacity], h_counts[n_batch].
 * The first call allocates a device scratch arena owned by the plan (FDAS_E_NOMEM on
 * failure); the call synchronises `stream` before returning. */
int fdas_search_host(fdas_plan* plan, const float* h_series, int32_t n_batch, int32_t max_harm,
                     const float* h_thresholds, fdas_cand* h_cands, uint32_t* h_counts,
                     uint32_t capacity, void* stream);

/* T_H with Q(H, T_H) = exp(-T) sum_{j<H} T^j/j! = pfa: the per-stage threshold for a
 * false-alarm probability pfa "under chi-squared statistics with 2H degrees of freedom"
 * (BJ:configs[4]). Host computation in fp64; returns NaN for H < 1 or pfa outside (0,1). */
double fdas_threshold(int32_t n_harm, double pfa);

/* Measurement aid: the FP32 fused-multiply-add rate of the current device in
 * TFLOP/s, from a kernel of independent FFMA chains (a <- a*x + y) on every SM, best of 4 timed
 * launches with CUDA events on `stream`; *out_ms (may be NULL) receives that launch's duration.
 * packed = 1 selects the same chains written with the packed f32x2 instruction of sm_100 (FFMA2, two
 * FMAs per lane and issue slot) so that both rates can be reported.
 * bench.py reports the fused correlate kernel against this measured peak as well as the nominal one.
 * Synchronises `stream`; allocates and frees 4 bytes of device memory.  Not part of the search path. */
int fdas_measure_fp32_tflops(double* out_tflops, double* out_ms, int32_t packed, void* stream);

/* Measurement aid: L2 -> SM read bandwidth in GB/s.  Every CTA (4 per SM) streams the same `bytes`-byte buffer
 * (1 MB .. 96 MB: L2-resident, far larger than L1) once with coalesced 16-byte loads; best of 3 timed launches with
 * CUDA events on `stream`.  bench.py reports the harmonic sum's inherent L2 -> SM stream (5.84 x the plane, DESIGN.md
 * section 6.3) against it.  Synchronises `stream`; allocates and frees `bytes` of device memory.  Not part of the search path. */
int fdas_measure_l2_gbs(double* out_gbs, size_t bytes, void* stream);

/* Measurement aid (the occupancy figures DESIGN.md section 6 quotes, from the runtime instead of by hand): resident
 * CTAs per SM (cudaOccupancyMaxActiveBlocksPerMultiprocessor), registers per thread and static + dynamic shared
 * memory per CTA of the BASELINE.json configs[2]/[4] instance of a kernel family on the current device.  kernel:
 * "spec_pass_a", "spec_pass_b", "spec_pass_c", "correlate", "correlate_fused", "correlate_staged", "harmsum"
 * (FDAS_E_INVALID otherwise).  Not part of the search path. */
int fdas_kernel_occupancy(const char* kernel, int32_t* ctas_per_sm, int32_t* registers, int32_t* smem_bytes);

int fdas_plan_destroy(fdas_plan* plan);

/* Static text for an FDAS_E_* code; for FDAS_E_CUDA the text of the last CUDA error seen. */
const char* fdas_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* FDAS_H */

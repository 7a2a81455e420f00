/*
 * fdas_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, fp64 CPU statement of what the FDAS hot path of arXiv
 * 1511.07343 computes (PAPER.md = the paper text).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call it.  It shares no code, header, table or helper with the CUDA path
 * under paper_1511_07343_b200/csrc/.
 *
 * What each function follows:
 *   ofdas_fft            textbook iterative radix-2 DFT, sign -1 forward (reading G6)
 *   ofdas_dft_direct     the O(n^2) definition  F_k = sum_n x_n e^{-2 pi i k n / N}
 *   ofdas_spectrum       PAPER.md:49 step 2 + BASELINE.json configs[0] ("keep bins
 *                        1..N/2, normalise by sqrt(mean |F_k|^2)")       [O1]
 *   ofdas_response       the constant-fdot Fourier response the paper cites from
 *                        Ransom et al. evaluated as the DFT of a
 *                        sampled linear-drift chirp                       [O2]
 *   ofdas_templates      T_z[j] = conj R_z(d_j), "complex conjugate
 *                        of the filter"                                   [O3]
 *   ofdas_correlate_direct   Eq. (1), as the direct sum      [O4]
 *   ofdas_correlate_fft  PAPER.md:49 steps 3-7 (overlap-save) with
 *                        this file's own FFT -- secondary, admitted only after it
 *                        matches the direct sum (tests/test_oracle_pins.py) [O7]
 *   ofdas_candidates     cells with P > threshold (BASELINE.json configs[0]) [O5]
 *   ofdas_harmsum        BASELINE.json configs[4]: S_H = sum_h P[z h/H, r h/H],
 *                        nearest grid point, integer-exact rounding       [O6]
 *   ofdas_threshold      Q(H, T) = e^-T sum_{j<H} T^j/j! = pfa (chi^2, 2H dof)
 *
 * Pins: tests/test_oracle_pins.py (P1..P13 of DESIGN.md).  The harmonic sum is pinned by its
 * index rule (P12) and by the closed form for a noise-free pulse train (P13); its statistics
 * on real pulsar data are outside what the paper fixes (paper silent) and stay unpinned.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

typedef struct {
    int32_t col;
    int16_t zi;
    int16_t nharm;
    double power;
} ofdas_cand;

static const double TWO_PI = 6.283185307179586476925286766559;

/* ---------------------------------------------------------------- FFT ---- */

/* In-place iterative radix-2 Cooley-Tukey, n a power of two.
 * sign = -1: forward  sum_n a_n e^{-2 pi i k n / n};  sign = +1: unnormalised inverse. */
int ofdas_fft(cplx *a, int64_t n, int sign)
{
    if (n < 1 || (n & (n - 1))) return -1;
    /* bit-reversal permutation */
    for (int64_t i = 1, j = 0; i < n; i++) {
        int64_t bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = a[i]; a[i] = a[j]; a[j] = t; }
    }
    for (int64_t len = 2; len <= n; len <<= 1) {
        int64_t half = len >> 1;
        cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)half);
        if (!w) return -2;
        for (int64_t j = 0; j < half; j++) {
            double ang = sign * TWO_PI * (double)j / (double)len;
            w[j] = cos(ang) + I * sin(ang);
        }
        #pragma omp parallel for schedule(static) if (n >= (1 << 16))
        for (int64_t i = 0; i < n; i += len) {
            for (int64_t j = 0; j < half; j++) {
                cplx u = a[i + j], v = a[i + j + half] * w[j];
                a[i + j] = u + v;
                a[i + j + half] = u - v;
            }
        }
        free(w);
    }
    return 0;
}

/* Serial version for use inside parallel regions (segments). */
static void fft_serial(cplx *a, int64_t n, int sign, const cplx *wtab /* n/2 entries e^{sign 2 pi i j/n} */)
{
    for (int64_t i = 1, j = 0; i < n; i++) {
        int64_t bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = a[i]; a[i] = a[j]; a[j] = t; }
    }
    (void)sign;
    for (int64_t len = 2; len <= n; len <<= 1) {
        int64_t half = len >> 1, stride = n / len;
        for (int64_t i = 0; i < n; i += len)
            for (int64_t j = 0; j < half; j++) {
                cplx u = a[i + j], v = a[i + j + half] * wtab[j * stride];
                a[i + j] = u + v;
                a[i + j + half] = u - v;
            }
    }
}

/* The O(n^2) definition, for pinning ofdas_fft on small n. */
void ofdas_dft_direct(const cplx *x, cplx *out, int64_t n, int sign)
{
    #pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; k++) {
        cplx acc = 0;
        for (int64_t j = 0; j < n; j++) {
            int64_t kj = (k * j) % n;              /* exact phase reduction */
            double ang = sign * TWO_PI * (double)kj / (double)n;
            acc += x[j] * (cos(ang) + I * sin(ang));
        }
        out[k] = acc;
    }
}

/* ----------------------------------------------------------- spectrum ---- */

/* O1.  x: float32[N] widened to double.  F = DFT_N(x) (forward, unnormalised);
 * keep k = 1..N/2 (drop DC, keep Nyquist): S[c] = F[c+1]/sqrt(mu),
 * mu = mean_{k=1..N/2} |F_k|^2.   F_raw (optional, N/2+1 entries k=0..N/2) gets
 * the un-normalised bins for the Parseval pin.  Degenerate case (paper silent; DESIGN.md
 * reading G22): a series whose kept bins are all exactly zero has mu = 0 and S := 0. */
int ofdas_spectrum(const float *x, int64_t N, cplx *S, double *mu_out, cplx *F_raw)
{
    if (N < 4 || (N & (N - 1))) return -1;
    cplx *a = (cplx *)malloc(sizeof(cplx) * (size_t)N);
    if (!a) return -2;
    for (int64_t i = 0; i < N; i++) a[i] = (double)x[i];
    int rc = ofdas_fft(a, N, -1);
    if (rc) { free(a); return rc; }
    int64_t nb = N / 2;
    double acc = 0.0;
    for (int64_t k = 1; k <= nb; k++) acc += creal(a[k]) * creal(a[k]) + cimag(a[k]) * cimag(a[k]);
    double mu = acc / (double)nb;
    double s = mu > 0.0 ? 1.0 / sqrt(mu) : 0.0;
    for (int64_t c = 0; c < nb; c++) S[c] = a[c + 1] * s;
    if (F_raw) for (int64_t k = 0; k <= nb; k++) F_raw[k] = a[k];
    if (mu_out) *mu_out = mu;
    free(a);
    return 0;
}

/* ---------------------------------------------------------- templates ---- */

/* O2.  R_z(d) = int_0^1 exp(2 pi i [(-d - z/2) u + (z/2) u^2]) du : the normalised
 * Fourier response, at offset d bins from the MEAN frequency, of a unit-amplitude
 * chirp drifting by z bins over the span (readings G1, G2, G5).
 * Evaluated as the DFT at bin K+d of the chirp of mean frequency K sampled at
 * n_t points u_n = (n + 1/2)/n_t (mid-point sampling: the left-point sum has an
 * O(1/n_t) end-point error at half-integer d where f(1) = -f(0); reading R2).
 * Phase is held in cycles and reduced mod 1 before sin/cos. */
void ofdas_response(double z, double d, int64_t n_t, double *re, double *im)
{
    double sr = 0.0, si = 0.0;
    double a = -d - 0.5 * z, b = 0.5 * z;
    for (int64_t n = 0; n < n_t; n++) {
        double u = ((double)n + 0.5) / (double)n_t;
        double cyc = a * u + b * u * u;
        cyc -= floor(cyc);
        sr += cos(TWO_PI * cyc);
        si += sin(TWO_PI * cyc);
    }
    *re = sr / (double)n_t;
    *im = si / (double)n_t;
}

/* O3.  Bank layout: template t = zi*(1+interbin) + s, z_zi = -z_max + zi*dz;
 * set s=0: offsets d_j = j - m/2; set s=1 (interbin): d_j = j - m/2 + 1/2.
 * T[t*m + j] = conj R_z(d_j).  No renormalisation (G11). */
int ofdas_templates(double z_max, double dz, int32_t m, int32_t interbin, int64_t n_t, cplx *T)
{
    int32_t n_z = (int32_t)llround(2.0 * z_max / dz) + 1;
    int32_t nset = 1 + (interbin ? 1 : 0);
    #pragma omp parallel for collapse(2) schedule(dynamic, 8)
    for (int32_t t = 0; t < n_z * nset; t++)
        for (int32_t j = 0; j < m; j++) {
            int32_t zi = t / nset, s = t % nset;
            double z = -z_max + zi * dz;
            double d = (double)(j - m / 2) + 0.5 * s;
            double re, im;
            ofdas_response(z, d, n_t, &re, &im);
            T[(int64_t)t * m + j] = re - I * im;
        }
    return n_z * nset;
}

/* -------------------------------------------------------- correlation ---- */

/* O4, Eq. (1) as the direct sum, for plane columns of bins c in [c0, c0+nc).
 *   integer set:  C_z[c]  = sum_j S[c + j - m/2]     T_z[j]
 *   half-bin set: C'_z[c] = sum_j S[c + j - m/2 + 1] T'_z[j]     (G12)
 * S = 0 outside [0, n_bins) (G9).  P[zi*ld + (c-c0)*nset + s] = |C|^2, ld = nc*nset. */
void ofdas_correlate_direct(const cplx *S, int64_t n_bins, const cplx *T, int32_t n_z, int32_t m,
                            int32_t interbin, int64_t c0, int64_t nc, double *P)
{
    int32_t nset = 1 + (interbin ? 1 : 0);
    int64_t ld = nc * nset;
    /* local zero-padded copy of the spectrum the columns need, split re/im */
    int64_t lo = c0 - m / 2, len = nc + m + 1;
    double *sr = (double *)calloc((size_t)len, sizeof(double));
    double *si = (double *)calloc((size_t)len, sizeof(double));
    for (int64_t i = 0; i < len; i++) {
        int64_t c = lo + i;
        if (c >= 0 && c < n_bins) { sr[i] = creal(S[c]); si[i] = cimag(S[c]); }
    }
    #pragma omp parallel for collapse(2) schedule(static)
    for (int32_t t = 0; t < n_z * nset; t++)
        for (int64_t blk = 0; blk < nc; blk += 4096) {
            int32_t zi = t / nset, s = t % nset;
            const cplx *Tz = T + (int64_t)t * m;
            int64_t hi = blk + 4096 < nc ? blk + 4096 : nc;
            for (int64_t c = blk; c < hi; c++) {
                double ar = 0.0, ai = 0.0;
                const double *pr = sr + c + s, *pi = si + c + s;
                for (int32_t j = 0; j < m; j++) {
                    double tr = creal(Tz[j]), ti = cimag(Tz[j]);
                    ar += pr[j] * tr - pi[j] * ti;
                    ai += pr[j] * ti + pi[j] * tr;
                }
                P[(int64_t)zi * ld + c * nset + s] = ar * ar + ai * ai;
            }
        }
    free(sr); free(si);
}

/* O7, PAPER.md:49 steps 3-7: overlap-save with segment length L and `step` kept
 * outputs per segment (step <= L - m, so the half-bin set fits too; G13).
 *   window  w[i] = S[s*step - m/2 + i], i in [0, L)
 *   filter  g[(-j) mod L] = T[j]  (integer set),  g'[(-(j+1)) mod L] = T'[j]  (half-bin set)
 *   y = IFFT_L( FFT_L(w) . FFT_L(g)/L ), first `step` outputs kept, rest discarded.
 * Full plane P[zi*n_cols + c*nset + s]. */
int ofdas_correlate_fft(const cplx *S, int64_t n_bins, const cplx *T, int32_t n_z, int32_t m,
                        int32_t interbin, int32_t L, int32_t step, double *P)
{
    int32_t nset = 1 + (interbin ? 1 : 0), n_t = n_z * nset;
    if (L < 2 || (L & (L - 1)) || step < 1 || step > L - m) return -1;
    int64_t n_cols = n_bins * nset;
    int64_t n_seg = (n_bins + step - 1) / step;
    cplx *wf = (cplx *)malloc(sizeof(cplx) * (size_t)(L / 2));
    cplx *wi = (cplx *)malloc(sizeof(cplx) * (size_t)(L / 2));
    cplx *W = (cplx *)malloc(sizeof(cplx) * (size_t)n_t * L);
    if (!wf || !wi || !W) return -2;
    for (int32_t j = 0; j < L / 2; j++) {
        double ang = TWO_PI * (double)j / (double)L;
        wf[j] = cos(ang) - I * sin(ang);
        wi[j] = cos(ang) + I * sin(ang);
    }
    for (int32_t t = 0; t < n_t; t++) {
        cplx *g = W + (int64_t)t * L;
        int32_t s = t % nset;
        memset(g, 0, sizeof(cplx) * (size_t)L);
        for (int32_t j = 0; j < m; j++) g[((L - j - s) % L + L) % L] = T[(int64_t)t * m + j];
        fft_serial(g, L, -1, wf);
        for (int32_t k = 0; k < L; k++) g[k] /= (double)L;
    }
    #pragma omp parallel
    {
        cplx *X = (cplx *)malloc(sizeof(cplx) * (size_t)L);
        cplx *Y = (cplx *)malloc(sizeof(cplx) * (size_t)L);
        #pragma omp for schedule(dynamic, 1)
        for (int64_t sg = 0; sg < n_seg; sg++) {
            int64_t base = sg * step - m / 2;
            for (int32_t i = 0; i < L; i++) {
                int64_t c = base + i;
                X[i] = (c >= 0 && c < n_bins) ? S[c] : 0.0;
            }
            fft_serial(X, L, -1, wf);
            for (int32_t t = 0; t < n_t; t++) {
                const cplx *Wt = W + (int64_t)t * L;
                for (int32_t k = 0; k < L; k++) Y[k] = X[k] * Wt[k];
                fft_serial(Y, L, +1, wi);
                int32_t zi = t / nset, s = t % nset;
                for (int32_t o = 0; o < step; o++) {
                    int64_t c = sg * step + o;
                    if (c >= n_bins) break;
                    double re = creal(Y[o]), im = cimag(Y[o]);
                    P[(int64_t)zi * n_cols + c * nset + s] = re * re + im * im;
                }
            }
        }
        free(X); free(Y);
    }
    free(wf); free(wi); free(W);
    return 0;
}

/* --------------------------------------------------------- candidates ---- */

/* O5.  All cells with P > thr (strict, G14); nharm = 1.  Returns the true count;
 * at most `cap` records are written, in row-major scan order. */
int64_t ofdas_candidates(const double *P, int32_t n_z, int64_t n_cols, double thr,
                         ofdas_cand *out, int64_t cap)
{
    int64_t n = 0;
    for (int32_t zi = 0; zi < n_z; zi++)
        for (int64_t c = 0; c < n_cols; c++) {
            double p = P[(int64_t)zi * n_cols + c];
            if (p > thr) {
                if (out && n < cap) { out[n].col = (int32_t)c; out[n].zi = (int16_t)zi; out[n].nharm = 1; out[n].power = p; }
                n++;
            }
        }
    return n;
}

/* O6.  Harmonic sum on an integer-bin plane.  True bin k = bin0 + col; signed
 * z index zeta = zi - zc, zc = (n_z-1)/2.  For H in {1,2,4,..,max_harm}, h = 1..H:
 *   k_h    = floor((k h + H/2)/H)                 (round half up, exact integers)
 *   zeta_h = sgn(zeta) floor((|zeta| h + H/2)/H)  (round half away from zero)
 *   S_H(k, zeta) = sum_h P[zc + zeta_h][k_h - bin0],  terms with k_h < bin0 contribute 0.
 * Candidate iff S_H > thr[log2 H] (strict).  S_out (optional): n_stage planes of S_H
 * (n_stage*n_z*n_cols doubles) for value parity.  Returns the true count. */
int64_t ofdas_harmsum(const double *P, int32_t n_z, int64_t n_cols, int32_t bin0, int32_t max_harm,
                      const double *thr, ofdas_cand *out, int64_t cap, double *S_out)
{
    int32_t zc = (n_z - 1) / 2;
    int64_t n = 0;
    int stage = 0;
    double *row = (double *)malloc(sizeof(double) * (size_t)n_cols);
    if (!row) return -2;
    for (int32_t H = 1; H <= max_harm; H <<= 1, stage++) {
        for (int32_t zi = 0; zi < n_z; zi++) {
            int32_t zeta = zi - zc, az = zeta < 0 ? -zeta : zeta, sg = zeta < 0 ? -1 : 1;
            #pragma omp parallel for schedule(static)
            for (int64_t c = 0; c < n_cols; c++) {
                int64_t k = (int64_t)bin0 + c;
                double acc = 0.0;
                for (int32_t h = 1; h <= H; h++) {
                    int64_t kh = (k * h + H / 2) / H;
                    int32_t zh = sg * (int32_t)(((int64_t)az * h + H / 2) / H);
                    if (kh < bin0) continue;
                    acc += P[(int64_t)(zc + zh) * n_cols + (kh - bin0)];
                }
                row[c] = acc;
            }
            if (S_out) memcpy(S_out + ((int64_t)stage * n_z + zi) * n_cols, row, sizeof(double) * (size_t)n_cols);
            if (thr)
                for (int64_t c = 0; c < n_cols; c++)
                    if (row[c] > thr[stage]) {
                        if (out && n < cap) { out[n].col = (int32_t)c; out[n].zi = (int16_t)zi; out[n].nharm = (int16_t)H; out[n].power = row[c]; }
                        n++;
                    }
        }
    }
    free(row);
    return n;
}

/* Q(H, T) = e^{-T} sum_{j<H} T^j / j!  (survival function of Gamma(H,1); 2S ~ chi^2_{2H}). */
double ofdas_gamma_q(int32_t H, double T)
{
    double term = 1.0, sum = 1.0;
    for (int32_t j = 1; j < H; j++) { term *= T / (double)j; sum += term; }
    return exp(-T) * sum;
}

/* Threshold T_H with Q(H, T_H) = pfa, by bisection (Q is strictly decreasing in T). */
double ofdas_threshold(int32_t H, double pfa)
{
    double lo = 0.0, hi = 1.0;
    while (ofdas_gamma_q(H, hi) > pfa) hi *= 2.0;
    for (int it = 0; it < 200; it++) {
        double mid = 0.5 * (lo + hi);
        if (ofdas_gamma_q(H, mid) > pfa) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

/* ------------------------------------------------- time-domain resampling ---- */

/* Time-domain acceleration trial ("resampling the time series according to a time
 * offset caused by the constant acceleration, followed by a standard periodicity search"; the
 * paper gives no formula: DESIGN.md reading G23).  With u = n/N in [0,1) the time offset of a
 * constant acceleration, referred to mid-span, is beta (u^2 - u); a signal of mean frequency r0
 * drifting z bins has phase r0 [u + (z/2r0)(u^2 - u)], so the trial beta = z/(2 r0) turns it into
 * a pure tone at r0.  Output sample m (u' = m/N) takes the input sample nearest to the u that
 * solves  u + beta (u^2 - u) = u',  u = 2u' / [(1-beta) + sqrt((1-beta)^2 + 4 beta u')]
 * (the root that tends to u' as beta -> 0; no cancellation):
 *   y[m] = x[ min(N-1, floor(u N + 1/2)) ].
 * Each operation is a separately rounded IEEE fp64 operation (no contraction), in this order, so
 * that the index can be reproduced bit for bit.  |beta| < 1/2 required (monotone map). */
__attribute__((optimize("fp-contract=off")))
int ofdas_resample(const float *x, int64_t N, double beta, float *y)
{
    if (N < 2 || !(beta > -0.5 && beta < 0.5)) return -1;
    const double omb = 1.0 - beta, omb2 = omb * omb, fb = 4.0 * beta, dN = (double)N;
    #pragma omp parallel for schedule(static)
    for (int64_t m = 0; m < N; m++) {
        double up = (double)m / dN;
        double disc = omb2 + fb * up;
        double u = (2.0 * up) / (omb + sqrt(disc));
        int64_t n = (int64_t)floor(u * dN + 0.5);
        if (n > N - 1) n = N - 1;
        if (n < 0) n = 0;
        y[m] = x[n];
    }
    return 0;
}

/*
 * lofar_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE ONLY.
 *
 * A plain, slow, double-precision restatement of the hot path of
 * arXiv 1612.06592 ("Realtime processing of LOFAR data for the detection of
 * nano-second pulses from the Moon"): tied-array beamforming with per-sub-band
 * de-dispersion phases -> inverse polyphase filter bank (inverse DFT + 16-tap
 * synthesis FIR) -> amplitude threshold trigger.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header, table or
 * constant generator with the CUDA library under paper_1612_06592_b200/csrc,
 * and neither includes the other.
 *
 * Everything here follows the order of the paper's processing chain
 * (section 2: "station beams ... combined into multiple smaller
 * beams ... recovered by inversion of the PPF ... de-dispersed ... trigger"),
 * with the concrete instance fixed by BASELINE.json (configs[0], north_star)
 * and the readings A1..A20 / definitions O0..O8 of SURVEY.md section 8(c),
 * restated in DESIGN.md.  No blocking, no FFT, no fusion: direct sums only.
 *
 * Pins (tests/test_oracle_pins.py) check each function against closed forms,
 * library special cases (numpy.fft, scipy.signal.firwin), brute force on tiny
 * sizes and invariants; see DESIGN.md "Oracle pins".
 *
 * Index names: s station, p polarisation, b beam, d STEC trial, k sub-band
 * (absolute bin index 0..M/2-1), j = k - k0 index into the selected set,
 * q slice, r residue 0..M-1, M FFT size (1024), P taps per branch (16).
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_API __attribute__((visibility("default")))

static const double TWO_PI = 6.283185307179586476925286766559;
static const double PI = 3.141592653589793238462643383280;

/* Number of OpenMP threads the loops below may use (bench.py times the oracle on one core and on all). */
ORACLE_API void lofar_oracle_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

ORACLE_API int lofar_oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------
 * O0  Prototype low-pass filter (BASELINE.json:configs[0]: "16384-tap windowed
 * sinc, cutoff 1/1024, Kaiser beta=9"; reading A7: cutoff relative to Nyquist).
 *   h[j] = sinc((j - (L-1)/2)/M) * I0(beta*sqrt(1 - (2j/(L-1) - 1)^2)) / I0(beta),
 *   L = M*P, sinc(x) = sin(pi x)/(pi x), then scaled so that sum(h) = 1.
 * ------------------------------------------------------------------------- */
static double bessel_i0(double x)
{
    /* I0(x) = sum_{m>=0} ((x/2)^m / m!)^2, summed until the term vanishes. */
    double sum = 1.0, term = 1.0, half = 0.5 * x;
    for (int m = 1; m < 500; ++m) {
        term *= half / (double)m;
        double t2 = term * term;
        sum += t2;
        if (t2 < 1e-40 * sum) break;
    }
    return sum;
}

ORACLE_API void lofar_oracle_prototype(int M, int P, double beta, double *h)
{
    const int L = M * P;
    const double alpha = 0.5 * (double)(L - 1);
    const double i0b = bessel_i0(beta);
    double total = 0.0;
    for (int j = 0; j < L; ++j) {
        double x = ((double)j - alpha) / (double)M;
        double sinc = (x == 0.0) ? 1.0 : sin(PI * x) / (PI * x);
        double u = 2.0 * (double)j / (double)(L - 1) - 1.0;
        double arg = 1.0 - u * u;
        if (arg < 0.0) arg = 0.0;
        double win = bessel_i0(beta * sqrt(arg)) / i0b;
        h[j] = sinc * win;
        total += h[j];
    }
    for (int j = 0; j < L; ++j) h[j] /= total;
}

/* ---------------------------------------------------------------------------
 * O1  PPF analysis, direct form (models the station filter bank, PAPER.md:34
 * "filtered into sub-bands by a polyphase filter (PPF)").  Generator-side
 * model and the forward half of the round-trip pins; NOT on the GPU path.
 *   Y[m][k] = sum_{j=0}^{L-1} h[j] * x[m*M + j] * exp(-2 pi i k j / M),
 *   k = 0..M/2-1, m = 0..T-1;  x has (T+P-1)*M samples.
 * ------------------------------------------------------------------------- */
ORACLE_API void lofar_oracle_ppf_analysis(const double *x, int M, int P, const double *h,
                                          int T, double complex *Y /* [T][M/2] */)
{
    const int L = M * P, H = M / 2;
    double complex *tw = (double complex *)malloc(sizeof(double complex) * (size_t)M);
    for (int a = 0; a < M; ++a) tw[a] = cexp(-I * TWO_PI * (double)a / (double)M);
#pragma omp parallel for collapse(2) schedule(static)
    for (int m = 0; m < T; ++m)
        for (int k = 0; k < H; ++k) {
            double complex acc = 0.0;
            for (int j = 0; j < L; ++j)
                acc += h[j] * x[(size_t)m * M + j] * tw[(int)(((long long)k * j) % M)];
            Y[(size_t)m * H + k] = acc;
        }
    free(tw);
}

/* ---------------------------------------------------------------------------
 * O3  Tables (BASELINE.json:north_star: "w[b,s,sb] = exp(i(2 pi f_sb tau_{b,s}
 * - phi_disp(f_sb)))", configs[0]: "phi(f) = 2 pi * 1.343e9 * STEC / f rad").
 *   f_sb(k)  = f_zone + k * clock/M                      (reading A1)
 *   W[b][s][j]  = exp(+2 pi i f_sb(k0+j) tau[b][s])      (reading A3)
 *   Dph[d][j]   = exp(-2 pi i * 1.343e9 * STEC_d / f_sb(k0+j))
 * ------------------------------------------------------------------------- */
ORACLE_API void lofar_oracle_tables(int S, int B, int D, int K, int k0, int M,
                                    double clock_hz, double f_zone_hz,
                                    const double *tau /* [B][S] seconds */,
                                    const double *stec /* [D] TECU */,
                                    double complex *W /* [B][S][K] */,
                                    double complex *Dph /* [D][K] */)
{
    for (int j = 0; j < K; ++j) {
        double f = f_zone_hz + (double)(k0 + j) * (clock_hz / (double)M);
        for (int b = 0; b < B; ++b)
            for (int s = 0; s < S; ++s) {
                double turns = f * tau[b * S + s];
                turns -= floor(turns);
                W[((size_t)b * S + s) * K + j] = cexp(I * TWO_PI * turns);
            }
        for (int d = 0; d < D; ++d) {
            double turns = 1.343e9 * stec[d] / f;
            turns -= floor(turns);
            Dph[(size_t)d * K + j] = cexp(-I * TWO_PI * turns);
        }
    }
}

/* Read one complex input sample.  X layout: [S][2][K][T][re,im], t fastest.
 * dtype 0 = int8, 1 = int16 ("native 16 bit integer format";
 * configs[2..4] use 8 bit). */
static inline double complex read_x(const void *X, int dtype, size_t idx)
{
    if (dtype == 0) {
        const int8_t *p = (const int8_t *)X + 2 * idx;
        return (double)p[0] + I * (double)p[1];
    } else {
        const int16_t *p = (const int16_t *)X + 2 * idx;
        return (double)p[0] + I * (double)p[1];
    }
}

/* ---------------------------------------------------------------------------
 * O4  Tied-array beamforming fused with the de-dispersion phase
 * ("the signal of each station has to be summed with a complex
 * weight given by the station position and the beam direction"
 * "multiplied in frequency domain by a complex weight depending on the ...
 * STEC"; readings A5, A9).
 *   Z[b][d][j][q] = Dph[d][j] * sum_s sum_p W[b][s][j] * X[s][p][j][q]
 * for slices q = q0 .. q0+nq-1 of a block holding T slices per row.
 * Output Z: [B*D][K][nq], series index = b*D + d.
 * ------------------------------------------------------------------------- */
ORACLE_API void lofar_oracle_beamform(const void *X, int dtype, int S, int K, long long T,
                                      int B, int D, const double complex *W,
                                      const double complex *Dph, long long q0, long long nq,
                                      double complex *Z)
{
#pragma omp parallel for collapse(2) schedule(static)
    for (int b = 0; b < B; ++b)
        for (int j = 0; j < K; ++j)
            for (long long q = 0; q < nq; ++q) {
                double complex acc = 0.0;
                for (int s = 0; s < S; ++s)
                    for (int p = 0; p < 2; ++p) {
                        size_t idx = (((size_t)s * 2 + p) * K + j) * (size_t)T + (size_t)(q0 + q);
                        acc += W[((size_t)b * S + s) * K + j] * read_x(X, dtype, idx);
                    }
                for (int d = 0; d < D; ++d)
                    Z[(((size_t)b * D + d) * K + j) * (size_t)nq + q] = Dph[(size_t)d * K + j] * acc;
            }
}

/* ---------------------------------------------------------------------------
 * O5  Naive Hermitian inverse DFT ("an inverse Fourier
 * transformation F^-1 y~ = y"; readings A10, A11: unnormalised, unselected
 * bins zero, bin M/2 zero, only Re of bin 0).
 *   y[q][r] = [k0==0] Re Z[0][q] + 2 * sum_{k in sel, k>=1} Re( Z[k][q] e^{+2 pi i k r / M} )
 * Z: one series, [K][nq] (row pitch nq).  y: [nq][M].
 * ------------------------------------------------------------------------- */
ORACLE_API void lofar_oracle_idft(const double complex *Z, int K, int k0, int M, long long nq,
                                  double *y)
{
    double complex *tw = (double complex *)malloc(sizeof(double complex) * (size_t)M);
    for (int a = 0; a < M; ++a) tw[a] = cexp(I * TWO_PI * (double)a / (double)M);
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < nq; ++q)
        for (int r = 0; r < M; ++r) {
            double acc = 0.0;
            for (int j = 0; j < K; ++j) {
                int k = k0 + j;
                double complex z = Z[(size_t)j * (size_t)nq + (size_t)q];
                if (k == 0)
                    acc += creal(z);
                else
                    acc += 2.0 * creal(z * tw[(int)(((long long)k * r) % M)]);
            }
            y[(size_t)q * M + r] = acc;
        }
    free(tw);
}

/* ---------------------------------------------------------------------------
 * O6  Direct-convolution polyphase synthesis (BASELINE.json:north_star
 * "16-tap polyphase synthesis filter with overlap carried across blocks";
 * reading A8: matched synthesis g = M*h, i.e. one application of H^T of the
 * paper's system H x^ = y; reading A12 for block edges).
 *   xhat[q*M + r] = M * sum_{t=0}^{P-1} h[r + t*M] * y[q - t][r]
 * ylead: [(P-1)+nq][M]; rows 0..P-2 are the P-1 slices before the window
 * (history of the previous block, zeros at stream start), rows P-1.. are the
 * window's own slices.  out: [nq*M].
 * ------------------------------------------------------------------------- */
ORACLE_API void lofar_oracle_synthesis(const double *ylead, int M, int P, const double *h,
                                       long long nq, double *out)
{
#pragma omp parallel for schedule(static)
    for (long long q = 0; q < nq; ++q)
        for (int r = 0; r < M; ++r) {
            double acc = 0.0;
            for (int t = 0; t < P; ++t)
                acc += h[r + t * M] * ylead[(size_t)(q + (P - 1) - t) * M + r];
            out[(size_t)q * M + r] = (double)M * acc;
        }
}

/* ---------------------------------------------------------------------------
 * O7  Envelope and sigma ("Triggering on the amplitude of a
 * pulse"; readings A13, A14).
 *   e[n]  = sqrt( (1/Wn) * sum_{j=0}^{Wn-1} x[n-j]^2 ),   Wn = 1 -> e = |x|
 *   sigma = sqrt( (1/N) * sum_{n=0}^{N-1} e[n]^2 )        over this block
 * xlead: [(Wn-1)+N]; the first Wn-1 samples precede the block (zeros at
 * stream start).  env: [N].  Returns sigma.
 * ------------------------------------------------------------------------- */
ORACLE_API double lofar_oracle_envelope(const double *xlead, long long N, int Wn, double *env)
{
    double total = 0.0;
    for (long long n = 0; n < N; ++n) {
        double acc = 0.0;
        for (int j = 0; j < Wn; ++j) {
            double v = xlead[n + (Wn - 1) - j];
            acc += v * v;
        }
        acc /= (double)Wn;
        env[n] = sqrt(acc);
        total += acc;
    }
    return sqrt(total / (double)N);
}

/* ---------------------------------------------------------------------------
 * O8  Candidates (BASELINE.json:configs: "trigger threshold 5 sigma of
 * envelope RMS"; configs[3]: "trigger reports the best trial per candidate";
 * reading A15).  For one beam with D trials:
 *   snr_d[n] = env[d][n] / sigma[d];  d* = argmax_d snr_d[n] (lowest d on ties);
 *   candidate iff snr_{d*}[n] > kappa (strict).
 * env: [D][N], sigma: [D].  Writes up to cap records (sample n, trial d*),
 * in increasing n.  Returns the true number of candidates.
 * ------------------------------------------------------------------------- */
ORACLE_API long long lofar_oracle_candidates(const double *env, const double *sigma, int D,
                                             long long N, double kappa, long long cap,
                                             long long *sample, int *trial)
{
    long long count = 0;
    for (long long n = 0; n < N; ++n) {
        int best = 0;
        double best_snr = env[n] / sigma[0];
        for (int d = 1; d < D; ++d) {
            double snr = env[(size_t)d * (size_t)N + (size_t)n] / sigma[d];
            if (snr > best_snr) { best_snr = snr; best = d; }
        }
        if (best_snr > kappa) {
            if (count < cap) { sample[count] = n; trial[count] = best; }
            ++count;
        }
    }
    return count;
}

/* ===========================================================================
 * Rows "next" of SURVEY.md section 8(f).  Same rules as above: plain, slow,
 * double precision, no code shared with the CUDA library.
 * =========================================================================== */

/* ---------------------------------------------------------------------------
 * O9  Causal sigma (f3; the ns-resolution signal is used "only
 * to trigger the read-out", so the threshold has to be known while the block
 * is being reconstructed).  Reading A21: the reference level of
 * block i is the envelope RMS of block i-1 of the same series,
 *   sigma_ref_i[s] = sigma_{i-1}[s]  (i >= 1),
 *   sigma_ref_0[s] = sigma_init[s] if the caller gave one, else sigma_0[s]
 *                    (the first block of a stream is its own reference),
 * and O8 is applied with sigma_ref in place of sigma.  The arithmetic of this
 * definition is O7 + O8 with another sigma argument; the state (sigma of the
 * previous block) is carried by the caller (oracle/lofar_oracle.py).
 * ------------------------------------------------------------------------- */

/* ---------------------------------------------------------------------------
 * O10  Time clustering of candidates into events (f3; what a read-out request
 * of the transient buffers needs).  Reading A22: input is the
 * candidate list of ONE block, one beam after the other, samples increasing
 * (O8's output order).  Consecutive candidates of the same beam belong to the
 * same event iff their samples differ by at most `gap`.  Per event:
 *   first, last sample; number of candidates; the peak = the candidate with
 *   the largest snr = env/sigma (the lowest sample on exact ties).
 * beam[n], sample[n], snr[n]: inputs.  ev_first/ev_last/ev_count/ev_peak
 * (index into the input list): outputs, capacity cap.  Returns the number of
 * events.
 * ------------------------------------------------------------------------- */
ORACLE_API long long lofar_oracle_cluster(const int *beam, const long long *sample, const double *snr,
                                          long long n, long long gap, long long cap,
                                          long long *ev_first, long long *ev_last, long long *ev_count,
                                          long long *ev_peak)
{
    long long nev = 0;
    long long i = 0;
    while (i < n) {
        long long j = i, peak = i;
        while (j + 1 < n && beam[j + 1] == beam[i] && sample[j + 1] - sample[j] <= gap) {
            ++j;
            if (snr[j] > snr[peak]) peak = j;
        }
        if (nev < cap) {
            ev_first[nev] = sample[i];
            ev_last[nev] = sample[j];
            ev_count[nev] = j - i + 1;
            ev_peak[nev] = peak;
        }
        ++nev;
        i = j + 1;
    }
    return nev;
}

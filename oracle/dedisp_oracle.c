/*
 * dedisp_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, obviously-correct fp64 CPU implementation of the channelised
 * overlap-save coherent dedispersion path of De & Gupta (arXiv:1509.00186),
 * written from PAPER.md.  It exists so that tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs can check and time the
 * CUDA path against something independent.  Nothing in the product
 * (paper_1509_00186_b200/) may include, link, import or call this file, and
 * this file shares no code, table or constant generator with the CUDA path.
 *
 * Citations: P:L<n> = /root/reference/PAPER.md line n.
 *
 * What it computes, step by step in the paper's order (Fig. 4):
 *   1. unpack int8 (re, im) voltage samples of one frequency channel
 *      ("real and imaginary parts ... 8-bit integers");
 *   2. forward FFT of length N over an N-sample segment;
 *   3. multiply by the chirp = taper x inverse transfer function
 *      (Eq. 3);
 *   4. inverse FFT;
 *   5. overlap-save: discard the samples polluted by the circular wrap of the
 *      impulse response, overlap the same number with the next segment
 *      (P:L125);
 *   6. square and integrate n_int samples.
 *
 * No blocking, fusion or reordering beyond the above.  The FFT is a textbook
 * iterative radix-2 (naive O(N^2) DFT when N <= 64).  Threading (pthreads) is
 * over independent channels only and does not change any arithmetic.
 *
 * Parity pins: every function here is pinned by tests/test_oracle_pins.py
 * (see DESIGN.md "Oracle pins"); nothing is "parity unpinned".
 *
 * Readings of the paper (DESIGN.md "Readings" R1..R13) that this file fixes:
 *   R1  chirp sign: Eq. 3 (printed exp(+2*pi*i*psi)) is the ISM's own
 *       in-band term -- the third term of Eq. 2 under H = exp(-i*phi), P:L107 --
 *       and "the transfer function to correct for the dispersion within the
 *       band is the inverse of the third term": the chirp applied is
 *       exp(-2*pi*i*psi), to the output of a forward DFT with kernel
 *       exp(-2*pi*i*k*n/N) of a band whose baseband frequency rises with sky
 *       frequency.  A negative DM entry applies Eq. 3 itself.
 *   R2  reference frequency of psi = the channel centre f_c, f in [-dv/2, dv/2).
 *   R3  f_c = F - B/2 + (c + 1/2) * dv.
 *   R5  bin k of the N-point FFT is baseband frequency k*dv/N for k < N/2 and
 *       (k - N)*dv/N for k >= N/2.
 *   R6  taper: none (default), Hann cos^2(pi f/dv), Welch 1 - (2f/dv)^2.
 *   R7  1/N on the inverse FFT.
 *   R8  D = 4.148808e15 Hz^2 s per pc cm^-3 (4.148808e9 in MHz/us units).
 *   R9  framing head/tail/L from the group delay of the applied filter.
 *   R10 int8 two's complement, re then im, layout [t][chan][2].
 *   R11 detection |v|^2 = re^2 + im^2; integration = plain sum of n_int samples.
 *   R12 no zero padding; output j covers input times head + j*n_int ...
 *   R16 sub-band alignment in whole output samples against the top channel (oracle_band_sum).
 *   R17 folding: bin = floor(frac(t/period) * n_bins) in fp64, sums and counts (oracle_fold).
 */
#include <complex.h>
#include <math.h>
#include <pthread.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* Dispersion constant, P:L117 (R8). */
#define ORACLE_D_HZ2_S 4.148808e15

typedef struct {
    int n_chan;          /* C */
    double bw_hz;        /* B */
    double f_center_hz;  /* F */
    int n_dm;
    const double *dm;    /* [n_dm], pc cm^-3, sign allowed (R1) */
    int n_fft;           /* N, power of two */
    int n_int;
    int taper;           /* 0 none, 1 Hann, 2 Welch (R6) */
} oracle_cfg_t;

/* ------------------------------------------------------------------ */
/* Transforms                                                          */
/* ------------------------------------------------------------------ */

/* Naive DFT straight from the definition:
 *   out[k] = sum_n in[n] * exp(sign * 2*pi*i*k*n / N),  sign = -1 forward, +1 inverse (no 1/N). */
void oracle_dft_naive(const double complex *in, double complex *out, int n, int sign)
{
    for (int k = 0; k < n; ++k) {
        double complex acc = 0.0;
        for (int m = 0; m < n; ++m) {
            /* reduce k*m mod n before forming the angle to keep it small */
            long long km = ((long long)k * m) % n;
            double ang = sign * 2.0 * M_PI * (double)km / (double)n;
            acc += in[m] * (cos(ang) + I * sin(ang));
        }
        out[k] = acc;
    }
}

/* Textbook in-place iterative radix-2 decimation-in-time FFT (bit-reversal
 * permutation, then log2 N butterfly stages).  Unnormalised.  n must be a
 * power of two.  sign = -1 forward, +1 inverse.  The stage twiddle
 * exp(sign*2*pi*i*k/len) is read from a per-thread table w[m] =
 * exp(-2*pi*i*m/n), m < n/2 (each entry one cos and one sin of the exact
 * angle), at m = k*(n/len); the inverse conjugates it. */
static void fft_radix2(double complex *x, int n, int sign)
{
    static __thread double complex *w = NULL;
    static __thread int w_n = 0;
    if (w_n != n) {
        free(w);
        w = malloc(sizeof(double complex) * (size_t)(n / 2 + 1));
        for (int m = 0; m < n / 2; ++m) {
            double ang = -2.0 * M_PI * (double)m / (double)n;
            w[m] = cos(ang) + I * sin(ang);
        }
        w_n = n;
    }
    /* bit reversal */
    for (int i = 1, j = 0; i < n; ++i) {
        int bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { double complex t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    for (int len = 2; len <= n; len <<= 1) {
        int half = len >> 1, step = n / len;
        for (int start = 0; start < n; start += len) {
            for (int k = 0; k < half; ++k) {
                double complex tw = sign < 0 ? w[k * step] : conj(w[k * step]);
                double complex u = x[start + k];
                double complex v = x[start + k + half] * tw;
                x[start + k] = u + v;
                x[start + k + half] = u - v;
            }
        }
    }
}

/* Public transform: naive DFT for n <= 64 (north_star: "a naive DFT for tiny
 * sizes, a textbook radix-2 FFT otherwise").  In place.  Returns 0, or -1 if n
 * is not a power of two (> 64). */
int oracle_fft(double complex *x, int n, int sign)
{
    if (n <= 0) return -1;
    if (n <= 64) {
        double complex tmp[64];
        oracle_dft_naive(x, tmp, n, sign);
        memcpy(x, tmp, sizeof(double complex) * (size_t)n);
        return 0;
    }
    if (n & (n - 1)) return -1;
    fft_radix2(x, n, sign);
    return 0;
}

/* Radix-2 forced (for the pin "FFT == brute-force DFT for all N <= 64"). */
int oracle_fft_radix2(double complex *x, int n, int sign)
{
    if (n <= 0 || (n & (n - 1))) return -1;
    fft_radix2(x, n, sign);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Frequencies, chirp (Eq. 3), taper                                   */
/* ------------------------------------------------------------------ */

/* Channel width dv = B / C (Nyquist resolution of a channel is 1/dv,
 * i.e. one complex sample per 1/dv seconds per channel). */
double oracle_chan_width(const oracle_cfg_t *cfg)
{
    return cfg->bw_hz / (double)cfg->n_chan;
}

/* Channel centre frequency (R3): channels tile [F - B/2, F + B/2) ascending. */
double oracle_chan_freq(const oracle_cfg_t *cfg, int c)
{
    double dv = oracle_chan_width(cfg);
    return cfg->f_center_hz - 0.5 * cfg->bw_hz + ((double)c + 0.5) * dv;
}

/* Baseband frequency of FFT bin k (R5). */
double oracle_bin_freq(const oracle_cfg_t *cfg, int k)
{
    double dv = oracle_chan_width(cfg);
    int n = cfg->n_fft;
    int ks = (k < n / 2) ? k : k - n;
    return (double)ks * dv / (double)n;
}

/* Chirp phase in CYCLES, Eq. 3 with f_o read as the channel centre
 * f_c (R2) and f_l as the offset f from it:
 *     psi = D * DM * f^2 / ((f + f_c) * f_c^2)
 * so that Eq. 3 reads exp(i * 2*pi * psi) (the ISM term; its inverse is applied, R1). */
double oracle_chirp_phase_cycles(double dm, double f_c_hz, double f_hz)
{
    return ORACLE_D_HZ2_S * dm * f_hz * f_hz / ((f_hz + f_c_hz) * f_c_hz * f_c_hz);
}

/* Taper (P:L123 names Hanning and Welch, no formula: R6). */
double oracle_taper(int taper, double f_hz, double dv_hz)
{
    if (taper == 1) { double c = cos(M_PI * f_hz / dv_hz); return c * c; }
    if (taper == 2) { double r = 2.0 * f_hz / dv_hz; return 1.0 - r * r; }
    return 1.0;
}

/* The chirp function of one (DM, channel): H[k] = taper * exp(-2*pi*i*psi),
 * psi the phase of Eq. 3 in cycles (the correction "is the inverse of
 * the third term in Equation 2", which Eq. 3 prints; "The taper
 * function multiplied with the inverse transfer function is known as the
 * chirp function"; sign R1). */
void oracle_chirp(const oracle_cfg_t *cfg, int d, int c, double complex *H)
{
    double dv = oracle_chan_width(cfg);
    double fc = oracle_chan_freq(cfg, c);
    for (int k = 0; k < cfg->n_fft; ++k) {
        double f = oracle_bin_freq(cfg, k);
        double psi = oracle_chirp_phase_cycles(cfg->dm[d], fc, f);
        psi -= floor(psi);                     /* reduce mod 1 cycle before trig */
        double ang = 2.0 * M_PI * psi;
        H[k] = oracle_taper(cfg->taper, f, dv) * (cos(ang) - I * sin(ang));
    }
}

/* ------------------------------------------------------------------ */
/* Overlap-save framing (R9)                                           */
/* ------------------------------------------------------------------ */

static long long roundup_ll(long long x, long long m) { return ((x + m - 1) / m) * m; }
static long long gcd_ll(long long a, long long b) { while (b) { long long t = a % b; a = b; b = t; } return a; }

/* D = "the length of the impulse response" = dispersion time in the band
 * (P:L121).  With the channel-centre reference (R2) the ISM (Eq. 3)
 * delays the low band edge against the centre by
 *     t_lo = D*|DM|*(1/(f_c - dv/2)^2 - 1/f_c^2)
 * and lets the high edge arrive early by
 *     t_hi = D*|DM|*(1/f_c^2 - 1/(f_c + dv/2)^2)          (delay law).
 * The applied filter exp(-2*pi*i*psi) has group delay +dpsi/df: for DM > 0 it
 * holds the high edge back by t_hi (an output sample needs PAST input: head)
 * and pulls the low edge forward by t_lo (needs FUTURE input: tail); for
 * DM < 0 the roles swap.  The worst case is the lowest channel.  One framing
 * for the whole plan:
 *     head  = roundup(n_head, n_int)
 *     D_tot = roundup(head + n_tail, lcm(32, n_int))
 *     tail  = D_tot - head,  L = N - D_tot
 * Returns 0, or -1 when head + tail >= N or L % n_int != 0. */
int oracle_framing(const oracle_cfg_t *cfg, int *head, int *tail, int *L)
{
    double dv = oracle_chan_width(cfg);
    long long need_head = 0, need_tail = 0;
    for (int c = 0; c < cfg->n_chan; ++c) {
        double fc = oracle_chan_freq(cfg, c);
        double lo = fc - 0.5 * dv, hi = fc + 0.5 * dv;
        for (int d = 0; d < cfg->n_dm; ++d) {
            double a = fabs(cfg->dm[d]);
            double t_lo = ORACLE_D_HZ2_S * a * (1.0 / (lo * lo) - 1.0 / (fc * fc));
            double t_hi = ORACLE_D_HZ2_S * a * (1.0 / (fc * fc) - 1.0 / (hi * hi));
            long long n_lo = (long long)ceil(t_lo * dv);
            long long n_hi = (long long)ceil(t_hi * dv);
            long long h = cfg->dm[d] >= 0.0 ? n_hi : n_lo;
            long long t = cfg->dm[d] >= 0.0 ? n_lo : n_hi;
            if (h > need_head) need_head = h;
            if (t > need_tail) need_tail = t;
        }
    }
    long long ni = cfg->n_int;
    long long lcm = 32 / gcd_ll(32, ni) * ni;
    long long hd = roundup_ll(need_head, ni);
    long long dtot = roundup_ll(hd + need_tail, lcm);
    long long tl = dtot - hd;
    long long len = (long long)cfg->n_fft - dtot;
    *head = (int)hd; *tail = (int)tl; *L = (int)len;
    if (len <= 0 || len % ni != 0) return -1;
    return 0;
}

/* In-band dispersion smear of one channel, seconds: D*DM*(f_lo^-2 - f_hi^-2)
 * (P:L39-41 delay law; "length of the response is equal to the
 * dispersion time in the observing band"). */
double oracle_smear_seconds(double dm, double f_lo_hz, double f_hi_hz)
{
    return ORACLE_D_HZ2_S * fabs(dm) * (1.0 / (f_lo_hz * f_lo_hz) - 1.0 / (f_hi_hz * f_hi_hz));
}

/* Transform-length rule: "the smallest power of 2 greater than
 * twice the number of samples corresponding to the dispersion time". */
long long oracle_nfft_rule(double smear_samples)
{
    long long n = 1;
    while ((double)n <= 2.0 * smear_samples) n <<= 1;
    return n;
}

/* Number of blocks / outputs for a one-shot call of T samples (R12). */
long long oracle_n_blocks(const oracle_cfg_t *cfg, long long T, int head, int tail, int L)
{
    (void)cfg;
    if (T < (long long)head + tail + L) return 0;
    return (T - head - tail) / L;
}

/* ------------------------------------------------------------------ */
/* The path itself                                                     */
/* ------------------------------------------------------------------ */

/* One (channel c, block b) unit, all DMs.
 *   in      int8 [T][C][2] time-major (R10)
 *   H       [n_dm][N] chirp of channel c
 *   out_blk [n_dm][L/n_int] integrated intensities of this block
 *   volt    optional [n_dm][L] dedispersed complex voltages of this block (may be NULL)
 * Steps 1-6 of the header, in order. */
static void unit_dedisp(const oracle_cfg_t *cfg, const int8_t *in, int c, long long b,
                        int head, int L, const double complex *H,
                        double complex *x, double complex *y,
                        double *out_blk, double complex *volt)
{
    int N = cfg->n_fft, C = cfg->n_chan, ni = cfg->n_int;
    int nout = L / ni;
    /* 1. unpack: block b reads input rows b*L .. b*L + N - 1 (overlap-save) */
    for (int n = 0; n < N; ++n) {
        const int8_t *p = in + (((long long)b * L + n) * C + c) * 2;
        x[n] = (double)p[0] + I * (double)p[1];
    }
    /* 2. forward FFT, kernel exp(-2 pi i k n / N) */
    oracle_fft(x, N, -1);
    for (int d = 0; d < cfg->n_dm; ++d) {
        /* 3. chirp multiply (Eq. 3) */
        for (int k = 0; k < N; ++k) y[k] = x[k] * H[(size_t)d * N + k];
        /* 4. inverse FFT with 1/N (R7) */
        oracle_fft(y, N, +1);
        for (int n = 0; n < N; ++n) y[n] /= (double)N;
        /* 5. keep n in [head, head + L) (overlap-save discard, R9) */
        if (volt) for (int n = 0; n < L; ++n) volt[(size_t)d * L + n] = y[head + n];
        /* 6. detect + integrate: plain sum of n_int squared moduli (R11) */
        for (int j = 0; j < nout; ++j) {
            double acc = 0.0;
            for (int i = 0; i < ni; ++i) {
                double complex v = y[head + j * ni + i];
                acc += creal(v) * creal(v) + cimag(v) * cimag(v);
            }
            out_blk[(size_t)d * nout + j] = acc;
        }
    }
}

typedef struct {
    const oracle_cfg_t *cfg; const int8_t *in; long long T; double *out; long long out_stride;
    int head, tail, L; long long nb; int c0, c1;
} chan_job_t;

static void *chan_worker(void *arg)
{
    chan_job_t *j = (chan_job_t *)arg;
    const oracle_cfg_t *cfg = j->cfg;
    int N = cfg->n_fft, nd = cfg->n_dm, nout = j->L / cfg->n_int;
    double complex *H = malloc(sizeof(double complex) * (size_t)nd * N);
    double complex *x = malloc(sizeof(double complex) * N);
    double complex *y = malloc(sizeof(double complex) * N);
    double *blk = malloc(sizeof(double) * (size_t)nd * nout);
    for (int c = j->c0; c < j->c1; ++c) {
        for (int d = 0; d < nd; ++d) oracle_chirp(cfg, d, c, H + (size_t)d * N);
        for (long long b = 0; b < j->nb; ++b) {
            unit_dedisp(cfg, j->in, c, b, j->head, j->L, H, x, y, blk, NULL);
            for (int d = 0; d < nd; ++d)
                memcpy(j->out + ((size_t)d * cfg->n_chan + c) * j->out_stride + (size_t)b * nout,
                       blk + (size_t)d * nout, sizeof(double) * nout);
        }
    }
    free(H); free(x); free(y); free(blk);
    return NULL;
}

/* Whole one-shot call.
 *   in   int8 [T][C][2];  out double [n_dm][C][out_stride], out_stride >= nb*L/n_int.
 * n_threads only splits the channel range; arithmetic per unit is unchanged.
 * Returns number of outputs per (dm, channel), or a negative error. */
long long oracle_dedisp(const oracle_cfg_t *cfg, const int8_t *in, long long T,
                        double *out, long long out_stride, int n_threads)
{
    int head, tail, L;
    if (oracle_framing(cfg, &head, &tail, &L)) return -1;
    long long nb = oracle_n_blocks(cfg, T, head, tail, L);
    long long nout = nb * (L / cfg->n_int);
    if (nout > out_stride) return -2;
    if (nb == 0) return 0;
    if (n_threads < 1) n_threads = 1;
    if (n_threads > cfg->n_chan) n_threads = cfg->n_chan;
    pthread_t *th = malloc(sizeof(pthread_t) * n_threads);
    chan_job_t *jobs = malloc(sizeof(chan_job_t) * n_threads);
    for (int t = 0; t < n_threads; ++t) {
        jobs[t] = (chan_job_t){cfg, in, T, out, out_stride, head, tail, L, nb,
                               (int)((long long)cfg->n_chan * t / n_threads),
                               (int)((long long)cfg->n_chan * (t + 1) / n_threads)};
        pthread_create(&th[t], NULL, chan_worker, &jobs[t]);
    }
    for (int t = 0; t < n_threads; ++t) pthread_join(th[t], NULL);
    free(th); free(jobs);
    return nout;
}

/* Sampled units, for checks at full BASELINE sizes: for each listed
 * (chan[i], block[i]) compute the [n_dm][L/n_int] outputs of that unit into
 * out_units[i][n_dm][L/n_int].  Same unit_dedisp as above.  Optionally the
 * complex voltages (volt_units[i][n_dm][L] as re,im pairs) when non-NULL. */
typedef struct {
    const oracle_cfg_t *cfg; const int8_t *in; const int *chan; const long long *block;
    double *out_units; double *volt_units; int head, L; int i0, i1;
} unit_job_t;

static void *unit_worker(void *arg)
{
    unit_job_t *j = (unit_job_t *)arg;
    const oracle_cfg_t *cfg = j->cfg;
    int N = cfg->n_fft, nd = cfg->n_dm, nout = j->L / cfg->n_int;
    double complex *H = malloc(sizeof(double complex) * (size_t)nd * N);
    double complex *x = malloc(sizeof(double complex) * N);
    double complex *y = malloc(sizeof(double complex) * N);
    int last_c = -1;
    for (int i = j->i0; i < j->i1; ++i) {
        int c = j->chan[i];
        if (c != last_c) { for (int d = 0; d < nd; ++d) oracle_chirp(cfg, d, c, H + (size_t)d * N); last_c = c; }
        double complex *volt = j->volt_units ? (double complex *)j->volt_units + (size_t)i * nd * j->L : NULL;
        unit_dedisp(cfg, j->in, c, j->block[i], j->head, j->L, H, x, y,
                    j->out_units + (size_t)i * nd * nout, volt);
    }
    free(H); free(x); free(y);
    return NULL;
}

long long oracle_dedisp_units(const oracle_cfg_t *cfg, const int8_t *in, long long T,
                              const int *chan, const long long *block, int n_units,
                              double *out_units, double *volt_units, int n_threads)
{
    int head, tail, L;
    if (oracle_framing(cfg, &head, &tail, &L)) return -1;
    long long nb = oracle_n_blocks(cfg, T, head, tail, L);
    for (int i = 0; i < n_units; ++i)
        if (chan[i] < 0 || chan[i] >= cfg->n_chan || block[i] < 0 || block[i] >= nb) return -3;
    if (n_threads < 1) n_threads = 1;
    if (n_threads > n_units) n_threads = n_units > 0 ? n_units : 1;
    pthread_t *th = malloc(sizeof(pthread_t) * n_threads);
    unit_job_t *jobs = malloc(sizeof(unit_job_t) * n_threads);
    for (int t = 0; t < n_threads; ++t) {
        jobs[t] = (unit_job_t){cfg, in, chan, block, out_units, volt_units, head, L,
                               (int)((long long)n_units * t / n_threads),
                               (int)((long long)n_units * (t + 1) / n_threads)};
        pthread_create(&th[t], NULL, unit_worker, &jobs[t]);
    }
    for (int t = 0; t < n_threads; ++t) pthread_join(th[t], NULL);
    free(th); free(jobs);
    return L / cfg->n_int;
}

/* Bit-exact unpack of one framed block (pin for the int8 path, R10):
 * dst[n] = (re, im) of in[b*L + n][c], n in [0, N). */
void oracle_unpack_block(const oracle_cfg_t *cfg, const int8_t *in, int c, long long b, int L,
                         double *dst_re_im)
{
    for (int n = 0; n < cfg->n_fft; ++n) {
        const int8_t *p = in + (((long long)b * L + n) * cfg->n_chan + c) * 2;
        dst_re_im[2 * n] = (double)p[0];
        dst_re_im[2 * n + 1] = (double)p[1];
    }
}

/* ---------------------------------------------------------------------------
 * NEXT-3: alignment of the coherently dedispersed
 * sub-bands in time and band sum.
 *
 * "Appropriate time delays are then applied to align the pulses in the
 * separate frequency channels, which are then added to produce a dedispersed
 * time series."  P:L67: "coherently dedispersing each sub-band, followed by
 * alignment of the individual sub-bands in time".
 *
 * Reading R16: after per-channel coherent dedispersion about the
 * channel centre, channel c carries the pulse at the arrival time of its
 * centre frequency f_c; relative to the highest channel it is late by
 *     delay(d, c) = D * DM_d * (1/f_c^2 - 1/f_top^2)          (P:L39-41 delay law)
 * seconds = delay * dv / n_int output samples.  Only whole output samples are
 * shifted ("time delays", not phase ramps):
 *     shift(d, c) = lround(delay * dv / n_int) - min_c' lround(...)   (>= 0, so a
 *                   negative DM, whose lowest channel arrives first, works too)
 *     series[d][j] = sum_c out[d][c][j + shift(d, c)],  j in [0, n_out - max_c shift)
 * ------------------------------------------------------------------------- */
void oracle_band_shifts(const oracle_cfg_t *cfg, int d, long long *shift /* [n_chan] */)
{
    double f_top = oracle_chan_freq(cfg, cfg->n_chan - 1);
    double dv = oracle_chan_width(cfg);
    long long lo = 0;
    for (int c = 0; c < cfg->n_chan; ++c) {
        double f_c = oracle_chan_freq(cfg, c);
        double delay_s = ORACLE_D_HZ2_S * cfg->dm[d] * (1.0 / (f_c * f_c) - 1.0 / (f_top * f_top));
        shift[c] = llround(delay_s * dv / (double)cfg->n_int);
        if (c == 0 || shift[c] < lo) lo = shift[c];
    }
    for (int c = 0; c < cfg->n_chan; ++c) shift[c] -= lo;
}

/* out [n_dm][n_chan][out_stride] (first n_out columns valid) -> series [n_dm][series_stride].
 * Returns n_series = n_out - (largest shift over all DMs and channels), the same length for every DM so that
 * the rows share a time axis; 0 if that is not positive. */
long long oracle_band_sum(const oracle_cfg_t *cfg, const double *out, long long out_stride, long long n_out,
                          double *series, long long series_stride)
{
    int C = cfg->n_chan;
    long long *shift = (long long *)malloc(sizeof(long long) * (size_t)C * cfg->n_dm);
    long long max_shift = 0;
    for (int d = 0; d < cfg->n_dm; ++d) {
        oracle_band_shifts(cfg, d, shift + (size_t)d * C);
        for (int c = 0; c < C; ++c)
            if (shift[(size_t)d * C + c] > max_shift) max_shift = shift[(size_t)d * C + c];
    }
    long long n_ser = n_out - max_shift;
    if (n_ser <= 0 || series_stride < n_ser) { free(shift); return 0; }
    for (int d = 0; d < cfg->n_dm; ++d)
        for (long long j = 0; j < n_ser; ++j) {
            double acc = 0.0;
            for (int c = 0; c < C; ++c)
                acc += out[((size_t)d * C + c) * out_stride + j + shift[(size_t)d * C + c]];
            series[(size_t)d * series_stride + j] = acc;
        }
    free(shift);
    return n_ser;
}

/* ---------------------------------------------------------------------------
 * NEXT-3, second half: folding a dedispersed time series into a pulse profile.
 * Every result figure of the paper is a folded profile (Figs. 1, 8, 13, 14;
 * P:L59) but the method is not described; reading R17
 * (DESIGN.md): sample j is taken at t_j = t0 + j*dt, its pulse phase is the
 * fractional part of t_j / period, it falls into bin floor(phase * n_bins)
 * (clamped to n_bins - 1), a bin's value is the SUM of its samples and the
 * number of samples per bin is returned beside it (profile = sum / count).
 * The bin decision is taken in fp64.
 * ------------------------------------------------------------------------- */
void oracle_fold(const double *series, long long n, double t0_s, double dt_s, double period_s, int n_bins,
                 double *sum /* [n_bins] */, long long *count /* [n_bins] */)
{
    for (int b = 0; b < n_bins; ++b) { sum[b] = 0.0; count[b] = 0; }
    for (long long j = 0; j < n; ++j) {
        double turns = (t0_s + (double)j * dt_s) / period_s;
        double phase = turns - floor(turns);
        int b = (int)(phase * (double)n_bins);
        if (b > n_bins - 1) b = n_bins - 1;
        sum[b] += series[j];
        count[b] += 1;
    }
}

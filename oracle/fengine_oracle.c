/*
 * fengine_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, float64 CPU statement of what the F-engine data path of
 * arxiv 2303.09886 ("Efficient channelization on a Graphics Processing Unit")
 * computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header, table or
 * constant with the CUDA path under paper_2303_09886_b200/.
 *
 * Every function cites the passage it follows as PAPER.md:<line> (section).
 * Readings of silent / ambiguous points are the R-numbers of DESIGN.md.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`):
 *   oracle_unpack10      P1  hand example + independent bit-by-bit packer round trip
 *   oracle_unpack_bits   P1b every code of 4/8/12/16-bit samples through an independent packer; b = 10 == oracle_unpack10
 *   oracle_window/fir    P2  impulse response, T=1 block FFT; P3 delay == input shift
 *   oracle_fft_radix2    P4  O(N^2) DFT, on-bin tone, Parseval (P6)
 *   whole path           P5  closed form for a tone (DTFT of h), P7, P8, P10, P12
 *   oracle_quantize      P9  rounding / saturation table
 * Absolute end-to-end values: the paper prints none -> "parity unpinned" beyond
 * the pins above.
 *
 * Build: gcc -O2 -std=c99 -fopenmp -shared -fPIC fengine_oracle.c -o libfengine_oracle.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_PI 3.14159265358979323846264338327950288

/* ---------------------------------------------------------------------------
 * O1  Unpack.  PAPER.md:31 (Sec 2.1 step 1: "10-bit signed integer voltage
 * samples"), PAPER.md:51 (Sec 2.2: 4096 samples = 5120 bytes, i.e. 4 samples in
 * 5 bytes).  Bit order (R1, BASELINE.json configs[0]): big-endian bit stream,
 * sample u occupies bits [10u, 10u+10), MSB first, two's complement.
 * ------------------------------------------------------------------------- */
static int unpack_one(const uint8_t *bytes, int64_t u)
{
    const uint8_t *b = bytes + 5 * (u >> 2);
    int v;
    switch ((int)(u & 3)) {
    case 0:  v = (b[0] << 2) | (b[1] >> 6); break;
    case 1:  v = ((b[1] & 63) << 4) | (b[2] >> 4); break;
    case 2:  v = ((b[2] & 15) << 6) | (b[3] >> 2); break;
    default: v = ((b[3] & 3) << 8) | b[4]; break;
    }
    return (v ^ 512) - 512;            /* sign-extend bit 9 */
}

void oracle_unpack10(const uint8_t *bytes, int64_t n_samples, int16_t *out)
{
    for (int64_t u = 0; u < n_samples; ++u)
        out[u] = (int16_t)unpack_one(bytes, u);
}

/* Other input bit depths (the paper's bit-depth sweep: "4, 8, 12 and 16-bit samples"): the same
 * convention as R1 with b bits per sample: big-endian bit stream, sample u in bits [b*u, b*u + b), MSB first, two's
 * complement.  Written bit by bit on purpose (no word tricks): b in 1..16. */
void oracle_unpack_bits(const uint8_t *bytes, int64_t n_samples, int bits, int16_t *out)
{
    for (int64_t u = 0; u < n_samples; ++u) {
        int v = 0;
        for (int i = 0; i < bits; ++i) {
            const int64_t bit = (int64_t)bits * u + i;
            v = (v << 1) | ((bytes[bit >> 3] >> (7 - (int)(bit & 7))) & 1);
        }
        if (v & (1 << (bits - 1))) v -= 1 << bits;      /* sign-extend */
        out[u] = (int16_t)v;
    }
}

/* ---------------------------------------------------------------------------
 * O2  Coarse delay as an index offset.  PAPER.md:32 (step 2)
 * (Eq. 1: index t0 + t - c + 2nj), PAPER.md:115 (Sec 3.3: "adjusting indices
 * used to fetch samples").  Spectrum m starts at t0 = N*m (R2), positive c
 * reads earlier samples (R4); samples outside [0, L) read as 0 (R3).
 * x[m'] = s[N*m - c + m'],  0 <= m' < N*T.
 * ------------------------------------------------------------------------- */
void oracle_window(const double *s, int64_t L, int N, int T, int64_t m, int64_t c, double *x)
{
    const int64_t u0 = (int64_t)N * m - c;
    for (int64_t i = 0; i < (int64_t)N * T; ++i) {
        const int64_t u = u0 + i;
        x[i] = (u >= 0 && u < L) ? s[u] : 0.0;
    }
}

/* ---------------------------------------------------------------------------
 * O3  PFB FIR, the direct sum of Eq. (1).  PAPER.md:33-35:
 *   g_t = sum_{j=0}^{T-1} s_{t0+t-c+2nj} * w_{t,j},   w_{t,j} = h[t + N*j]
 * (BASELINE.json configs[0] for the flat weight order; R5: no time reversal).
 * ------------------------------------------------------------------------- */
void oracle_fir(const double *x, const float *h, int N, int T, double *g)
{
    for (int t = 0; t < N; ++t) {
        double acc = 0.0;
        for (int j = 0; j < T; ++j)
            acc += x[t + (int64_t)N * j] * (double)h[t + (int64_t)N * j];
        g[t] = acc;
    }
}

/* ---------------------------------------------------------------------------
 * O4  Fourier transform.  PAPER.md:37: "a 2n-element real-to-complex Fourier
 * transform, from which only the n non-negative frequencies are retained";
 * forward sign, unnormalised (R8).  Textbook iterative radix-2 decimation in
 * time on the complex sequence (g, 0); twiddles exp(-2 pi i q / N) come from a
 * table filled by direct cos/sin per index (no recurrences).
 * oracle_dft is the O(N^2) definition, used for tiny N.
 * ------------------------------------------------------------------------- */
void oracle_twiddles(int N, double *tw_re, double *tw_im)   /* N/2 entries */
{
    for (int q = 0; q < N / 2; ++q) {
        const double ang = -2.0 * ORACLE_PI * (double)q / (double)N;
        tw_re[q] = cos(ang);
        tw_im[q] = sin(ang);
    }
}

void oracle_fft_radix2(double *re, double *im, int N, const double *tw_re, const double *tw_im)
{
    /* bit-reversal permutation */
    for (int i = 1, j = 0; i < N; ++i) {
        int bit = N >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = re[i]; re[i] = re[j]; re[j] = tr;
            double ti = im[i]; im[i] = im[j]; im[j] = ti;
        }
    }
    for (int len = 2; len <= N; len <<= 1) {
        const int half = len >> 1, step = N / len;
        for (int base = 0; base < N; base += len) {
            for (int q = 0; q < half; ++q) {
                const double wr = tw_re[q * step], wi = tw_im[q * step];
                const int a = base + q, b = a + half;
                const double xr = re[b] * wr - im[b] * wi;
                const double xi = re[b] * wi + im[b] * wr;
                re[b] = re[a] - xr; im[b] = im[a] - xi;
                re[a] = re[a] + xr; im[a] = im[a] + xi;
            }
        }
    }
}

void oracle_dft(const double *g, int N, int n_out, double *Xre, double *Xim)
{
    for (int k = 0; k < n_out; ++k) {
        double sr = 0.0, si = 0.0;
        for (int t = 0; t < N; ++t) {
            /* reduce k*t mod N in integers so the angle stays small and exact */
            const int64_t r = ((int64_t)k * t) % N;
            const double ang = -2.0 * ORACLE_PI * (double)r / (double)N;
            sr += g[t] * cos(ang);
            si += g[t] * sin(ang);
        }
        Xre[k] = sr; Xim[k] = si;
    }
}

/* ---------------------------------------------------------------------------
 * O7  Quantise.  PAPER.md:43 ("quantized to 8-bit signed Gaussian integers"),
 * PAPER.md:161 ("rounding and saturation").  Round half to even, then clamp to
 * [-127, 127]; NaN -> 0 (R11).
 * ------------------------------------------------------------------------- */
int oracle_quantize(double v)
{
    if (v != v) return 0;
    double r = nearbyint(v);            /* default FE_TONEAREST: ties to even */
    if (r > 127.0) r = 127.0;
    if (r < -127.0) r = -127.0;
    return (int)r;
}

/* ---------------------------------------------------------------------------
 * One (stream, spectrum): O2..O7 in order.
 *   X  = FFT_N(g)[0..n)
 *   R  = exp(i(-2 pi d k / N + phi))                 PAPER.md:41 (R9)
 *   Y  = (X * R) * G[k]                              PAPER.md:42 (R10)
 *   q  = clamp(rint(Y))
 * Yout (nullable): n complex doubles (re, im interleaved) for this stream and
 * spectrum; qout: n (re, im) int8 pairs; nyq (nullable): the dropped Nyquist
 * bin X[n] (re only is meaningful; im is 0 up to rounding), for Parseval.
 * ------------------------------------------------------------------------- */
static void one_spectrum(const double *s, int64_t L, int N, int T, const float *h,
                         int64_t m, int64_t c, double d, double phi, const float *G,
                         const double *tw_re, const double *tw_im, int use_dft,
                         double *x, double *re, double *im,
                         double *Yout, int ystride, int8_t *qout, int qstride, double *nyq)
{
    const int n = N / 2;
    oracle_window(s, L, N, T, m, c, x);
    oracle_fir(x, h, N, T, re);                 /* g in re[] */
    if (use_dft) {
        double *g = (double *)malloc(sizeof(double) * N);
        memcpy(g, re, sizeof(double) * N);
        oracle_dft(g, N, n + 1, re, im);
        free(g);
    } else {
        memset(im, 0, sizeof(double) * N);
        oracle_fft_radix2(re, im, N, tw_re, tw_im);
    }
    if (nyq) { nyq[0] = re[n]; nyq[1] = im[n]; }
    for (int k = 0; k < n; ++k) {
        const double ang = -2.0 * ORACLE_PI * d * (double)k / (double)N + phi;
        const double rr = cos(ang), ri = sin(ang);
        const double xr = re[k] * rr - im[k] * ri;          /* X * R */
        const double xi = re[k] * ri + im[k] * rr;
        const double gr = (double)G[2 * k], gi = (double)G[2 * k + 1];
        const double yr = xr * gr - xi * gi;                /* (X R) * G */
        const double yi = xr * gi + xi * gr;
        if (Yout) { Yout[(int64_t)k * ystride] = yr; Yout[(int64_t)k * ystride + 1] = yi; }
        if (qout) {
            qout[(int64_t)k * qstride]     = (int8_t)oracle_quantize(yr);
            qout[(int64_t)k * qstride + 1] = (int8_t)oracle_quantize(yi);
        }
    }
}

/* ---------------------------------------------------------------------------
 * Whole path on float64 samples (the entry the linearity and unquantised-tone
 * pins use).  Layouts:
 *   s       [A][P][L]            double, L = N*(S_total + T - 1) or any L
 *   h       [N*T]                float  (weights[t + N*j] = w[t][j])
 *   coarse  [A][P][n_coarse]     int32, n_coarse == 1 -> constant, else entry m
 *   fine_d, fine_phi [A][P][n_fine]  float, same rule
 *   gains   [A][P][n][2]         float (re, im)
 *   sel     [n_sel] spectrum indices to compute (NULL -> 0..n_sel-1)
 *   out     [A][n_sel][n][P][2]  int8      (both pols in one record;
 *                                           BASELINE.json configs[0] layout)
 *   Y       [A][n_sel][n][P][2]  double, nullable (pre-quantisation)
 *   nyq     [A][P][n_sel][2]     double, nullable (dropped Nyquist bin of X)
 * Returns 0, or 1 on invalid arguments.
 * ------------------------------------------------------------------------- */
int oracle_channelize_f64(int A, int n, int T, int P, const float *h,
                          const int32_t *coarse, int64_t n_coarse,
                          const float *fine_d, const float *fine_phi, int64_t n_fine,
                          const float *gains, const double *s, int64_t L,
                          const int64_t *sel, int64_t n_sel,
                          int8_t *out, double *Y, double *nyq, int use_dft, int n_threads)
{
    if (A < 1 || n < 1 || (n & (n - 1)) || T < 1 || P < 1 || P > 2 || n_sel < 0) return 1;
    const int N = 2 * n;
    double *tw_re = (double *)malloc(sizeof(double) * (N / 2 + 1));
    double *tw_im = (double *)malloc(sizeof(double) * (N / 2 + 1));
    oracle_twiddles(N, tw_re, tw_im);
    const int64_t n_units = (int64_t)A * P * n_sel;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
    #pragma omp parallel
    {
        double *x  = (double *)malloc(sizeof(double) * (size_t)N * T);
        double *re = (double *)malloc(sizeof(double) * N);
        double *im = (double *)malloc(sizeof(double) * N);
        #pragma omp for schedule(dynamic, 4)
        for (int64_t unit = 0; unit < n_units; ++unit) {
            const int64_t i = unit % n_sel;
            const int p = (int)((unit / n_sel) % P);
            const int a = (int)(unit / n_sel / P);
            const int64_t m = sel ? sel[i] : i;
            const int64_t st = (int64_t)a * P + p;
            const int64_t c = coarse ? coarse[st * n_coarse + (n_coarse == 1 ? 0 : m)] : 0;
            const double d   = fine_d   ? (double)fine_d  [st * n_fine + (n_fine == 1 ? 0 : m)] : 0.0;
            const double phi = fine_phi ? (double)fine_phi[st * n_fine + (n_fine == 1 ? 0 : m)] : 0.0;
            const int64_t rec = (((int64_t)a * n_sel + i) * n) * P * 2 + (int64_t)p * 2;
            one_spectrum(s + st * L, L, N, T, h, m, c, d, phi, gains + st * n * 2,
                         tw_re, tw_im, use_dft, x, re, im,
                         Y ? Y + rec : NULL, P * 2, out ? out + rec : NULL, P * 2,
                         nyq ? nyq + (st * n_sel + i) * 2 : NULL);
        }
        free(x); free(re); free(im);
    }
    free(tw_re); free(tw_im);
    return 0;
}

/* ---------------------------------------------------------------------------
 * Whole path on packed 10-bit input: O1 then the above.
 *   in   [A][P][L*5/4] bytes, L = N*(S_in + T - 1) with S_in = n_spectra_in.
 * ------------------------------------------------------------------------- */
int oracle_process(int A, int n, int T, int P, const float *h,
                   const int32_t *coarse, int64_t n_coarse,
                   const float *fine_d, const float *fine_phi, int64_t n_fine,
                   const float *gains, const uint8_t *in, int64_t n_spectra_in,
                   const int64_t *sel, int64_t n_sel,
                   int8_t *out, double *Y, double *nyq, int use_dft, int n_threads)
{
    if (A < 1 || n < 2 || T < 1 || P < 1 || n_spectra_in < 0) return 1;
    const int64_t L = (int64_t)2 * n * (n_spectra_in + T - 1);
    const int64_t n_streams = (int64_t)A * P;
    double *s = (double *)malloc(sizeof(double) * (size_t)(n_streams * L));
    if (!s) return 2;
    for (int64_t st = 0; st < n_streams; ++st) {
        const uint8_t *bytes = in + st * (L / 4 * 5);
        for (int64_t u = 0; u < L; ++u)
            s[st * L + u] = (double)unpack_one(bytes, u);
    }
    const int rc = oracle_channelize_f64(A, n, T, P, h, coarse, n_coarse, fine_d, fine_phi, n_fine,
                                         gains, s, L, sel, n_sel, out, Y, nyq, use_dft, n_threads);
    free(s);
    return rc;
}

/* ---------------------------------------------------------------------------
 * The definition written out for ONE output value (no FIR/FFT factorisation):
 *   X[k] = sum_{m'=0}^{NT-1} h[m'] * s[N*m - c + m'] * exp(-2 pi i k m' / N)
 * which equals Eq. (1) followed by the N-point transform because
 * exp(-2 pi i k (t + N j)/N) = exp(-2 pi i k t / N).
 * Then Y = X * R * G as above.  Used for sampled checks at full problem sizes
 * and as a structural cross-check of the FIR+FFT route (pin P12).
 * ------------------------------------------------------------------------- */
void oracle_direct_channel(const uint8_t *stream_bytes, int64_t L, int n, int T, const float *h,
                           int64_t m, int64_t c, double d, double phi, double g_re, double g_im,
                           int k, double *Yre, double *Yim)
{
    const int N = 2 * n;
    const int64_t u0 = (int64_t)N * m - c;
    double sr = 0.0, si = 0.0;
    for (int64_t i = 0; i < (int64_t)N * T; ++i) {
        const int64_t u = u0 + i;
        if (u < 0 || u >= L) continue;
        const double v = (double)unpack_one(stream_bytes, u) * (double)h[i];
        const int64_t r = ((int64_t)k * (i % N)) % N;
        const double ang = -2.0 * ORACLE_PI * (double)r / (double)N;
        sr += v * cos(ang);
        si += v * sin(ang);
    }
    const double ang = -2.0 * ORACLE_PI * d * (double)k / (double)N + phi;
    const double rr = cos(ang), ri = sin(ang);
    const double xr = sr * rr - si * ri, xi = sr * ri + si * rr;
    *Yre = xr * g_re - xi * g_im;
    *Yim = xr * g_im + xi * g_re;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/*
 * plspec_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, float64 CPU statement of the hot path of arXiv 2311.18737
 * ("GPGPU Acceleration of Incoherent Scatter Radar Plasma Line Analysis"):
 * spectral integration of coded radar echoes.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference leg may call this.  It shares no
 * code, header, table or helper with the CUDA path under paper_2311_18737_b200/csrc.
 *
 * What it computes (the definition itself; the method reaches it exactly up to rounding):
 *
 *   S[r][f] += sum_p | sum_{t<N} d_{p,r}[t] * exp(-2*pi*i*f*t/N) |^2
 *   d_{p,r}[t] = V[p][r0 + r*stride + t] * conj(C[p][t])   for t <  code_len
 *              = 0                                         for code_len <= t < N
 *
 * following, step by step, PAPER.md:83 (sec. 2.2): "a complex conjugation of the
 * transmit pulse, a complex multiplication of this into one range gate of the return
 * echo, and a Fourier transform of that result. We square this to arrive at the power
 * for the single range gate used. Repeating this by iterating through the number of
 * range gates we desire and the amount to step each of them", and PAPER.md:105-121
 * (sec. 3.2.1 complex multiplication, 3.2.2 FFT over rows of power-of-two length,
 * 3.2.3 spectrum accumulation "adding these to a new spectrum floating point array",
 * 3.2.4 looping over pulses "accumulating the results").
 *
 * Readings of the paper where it is silent:
 *   A1 forward transform, kernel exp(-2 pi i f t / N);  A2 un-normalised FFT, plain sum
 *   over pulses (no 1/N, no 1/P);  A3 "square" = squared modulus Re^2+Im^2 (Eq. 8,
 *   PAPER.md:79);  A4 conj on the transmit code only;  A5 echo index r0 + r*stride + t;
 *   A6 code_len <= N, zero padded;  A7 N a power of two;  A9 natural bin order, DC at 0;
 *   A11 one code per pulse;  A12 sc16 = interleaved int16 (I,Q), no scaling.
 *
 * The FFT is this file's own iterative radix-2 (bit reversal, then log2 N butterfly
 * stages); every twiddle is cos/sin(-2 pi k / N) evaluated directly in float64 (no
 * recurrence).  Pins (tests/test_oracle_pins.py): brute-force O(N^2) DFT, Parseval,
 * single-tone closed form (incl. Dirichlet kernel for code_len < N), identity code vs
 * numpy.fft, zero input, modulation / conjugation / scaling / gate-shift invariances.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libplspec_oracle.so plspec_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_CF32 0
#define ORACLE_SC16 1

static int is_pow2(int n) { return n >= 2 && (n & (n - 1)) == 0; }

/* In-place forward DFT of x (interleaved re,im; length N, power of two).
 * tw holds N/2 twiddles exp(-2 pi i k / N), interleaved. */
static void fft_radix2(double *x, int N, const double *tw)
{
    /* bit-reversal permutation */
    for (int i = 1, j = 0; i < N; i++) {
        int bit = N >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) {
            double tr = x[2 * i], ti = x[2 * i + 1];
            x[2 * i] = x[2 * j];
            x[2 * i + 1] = x[2 * j + 1];
            x[2 * j] = tr;
            x[2 * j + 1] = ti;
        }
    }
    /* log2 N decimation-in-time stages: len = 2, 4, ..., N */
    for (int len = 2; len <= N; len <<= 1) {
        int half = len >> 1;
        int step = N / len; /* twiddle index stride: exp(-2 pi i k/len) = tw[k*step] */
        for (int base = 0; base < N; base += len) {
            for (int k = 0; k < half; k++) {
                double wr = tw[2 * (k * step)], wi = tw[2 * (k * step) + 1];
                double *a = x + 2 * (base + k);
                double *b = x + 2 * (base + k + half);
                double br = b[0] * wr - b[1] * wi;
                double bi = b[0] * wi + b[1] * wr;
                b[0] = a[0] - br;
                b[1] = a[1] - bi;
                a[0] = a[0] + br;
                a[1] = a[1] + bi;
            }
        }
    }
}

static double *make_twiddles(int N)
{
    double *tw = (double *)malloc(sizeof(double) * (size_t)(N > 2 ? N : 2));
    if (!tw) return NULL;
    for (int k = 0; k < N / 2; k++) {
        double ang = -2.0 * M_PI * (double)k / (double)N;
        tw[2 * k] = cos(ang);
        tw[2 * k + 1] = sin(ang);
    }
    return tw;
}

/* Exposed so the FFT core can be pinned on its own against a brute-force DFT. */
int plspec_oracle_fft(double *x_interleaved, int N)
{
    if (!x_interleaved || !is_pow2(N)) return -1;
    double *tw = make_twiddles(N);
    if (!tw) return -2;
    fft_radix2(x_interleaved, N, tw);
    free(tw);
    return 0;
}

/* S[r][f] += sum over the n_ipp pulses given.  S is float64 [n_ranges][N], caller-owned,
 * caller-initialised (so several calls accumulate).
 * voltages: [n_ipp][ipp_len] complex64 (2 x float32) or sc16 (2 x int16), per dtype.
 * codes:    [n_ipp][code_len] complex64.
 * n_threads <= 0: OpenMP default.  Returns 0, or a negative value on a bad argument. */
int plspec_oracle_accumulate(int N, int code_len, int n_ranges, int r0, int stride,
                             int ipp_len, int dtype, const void *voltages,
                             const float *codes, int n_ipp, double *S, int n_threads)
{
    if (!is_pow2(N) || code_len < 1 || code_len > N || n_ranges < 1 || r0 < 0 ||
        stride < 1 || n_ipp < 0 || (dtype != ORACLE_CF32 && dtype != ORACLE_SC16))
        return -1;
    long long span = (long long)r0 + (long long)(n_ranges - 1) * stride + code_len;
    if (ipp_len == 0) ipp_len = (int)span;
    if (span > ipp_len) return -1;
    if (n_ipp == 0) return 0;
    if (!voltages || !codes || !S) return -1;

    double *tw = make_twiddles(N);
    if (!tw) return -2;
    int status = 0;
#ifdef _OPENMP
    if (n_threads > 0) omp_set_num_threads(n_threads);
#endif
#pragma omp parallel
    {
        double *d = (double *)malloc(sizeof(double) * 2 * (size_t)N);
        if (!d) {
#pragma omp critical
            status = -2;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int r = 0; r < n_ranges; r++) {              /* range gates */
                double *Srow = S + (size_t)r * N;
                for (int p = 0; p < n_ipp; p++) {             /* pulses     */
                    const float *c = codes + (size_t)p * code_len * 2;
                    size_t off = (size_t)p * ipp_len + (size_t)r0 + (size_t)r * stride;
                    for (int t = 0; t < code_len; t++) {      /* decode     */
                        double vr, vi;
                        if (dtype == ORACLE_CF32) {
                            const float *v = (const float *)voltages + 2 * (off + t);
                            vr = (double)v[0];
                            vi = (double)v[1];
                        } else {
                            const int16_t *v = (const int16_t *)voltages + 2 * (off + t);
                            vr = (double)v[0];
                            vi = (double)v[1];
                        }
                        double cr = (double)c[2 * t], ci = (double)c[2 * t + 1];
                        /* v * conj(c) */
                        d[2 * t] = vr * cr + vi * ci;
                        d[2 * t + 1] = vi * cr - vr * ci;
                    }
                    for (int t = code_len; t < N; t++) {      /* zero pad (reading A6)     */
                        d[2 * t] = 0.0;
                        d[2 * t + 1] = 0.0;
                    }
                    fft_radix2(d, N, tw);                     /* FFT        */
                    for (int f = 0; f < N; f++)               /* |X|^2, accumulate (:115)  */
                        Srow[f] += d[2 * f] * d[2 * f] + d[2 * f + 1] * d[2 * f + 1];
                }
            }
            free(d);
        }
    }
    free(tw);
    return status;
}

int plspec_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

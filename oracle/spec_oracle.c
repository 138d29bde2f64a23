/*
 * spec_oracle.c — CPU ORACLE (test infrastructure; see spec_oracle.h for scope and citations).
 * Plain C, double precision, written from PAPER.md section 4 (lines 59, 81-96) and the
 * readings listed in DESIGN.md section 3.  Shares nothing with the CUDA path.
 */
#include "spec_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846264338327950288
#endif

/* ------------------------------------------------------------------ coefficients */

static double sinc_pi(double x) /* sin(pi x)/(pi x), sinc(0)=1 */
{
    if (x == 0.0) return 1.0;
    return sin(M_PI * x) / (M_PI * x);
}

void oracle_default_coeffs(int nchan, int ntaps, int mode, int window, float *out)
{
    if (mode == ORACLE_MODE_FFT) {
        for (int k = 0; k < nchan; k++) {
            double w = 1.0;
            if (window == ORACLE_WINDOW_HANN) w = 0.5 * (1.0 - cos(2.0 * M_PI * (double)k / (double)nchan));
            out[k] = (float)w;
        }
        return;
    }
    long L = (long)ntaps * (long)nchan;
    for (long k = 0; k < L; k++) {
        /* (k - T*N/2)/N ; T*N/2 may be a half-integer multiple of N for odd T, keep it exact in double */
        double x = ((double)k - 0.5 * (double)L) / (double)nchan;
        double w = 1.0;
        if (window == ORACLE_WINDOW_HANN) w = 0.5 * (1.0 - cos(2.0 * M_PI * (double)k / (double)L));
        out[k] = (float)(sinc_pi(x) * w);
    }
}

/* ------------------------------------------------------------------ FIR */

void oracle_fir(int nchan, int ntaps, const double *h, const double *x, double *y)
{
    for (int n = 0; n < nchan; n++) {
        double re = 0.0, im = 0.0;
        for (int t = 0; t < ntaps; t++) {
            double c = h[(size_t)t * nchan + n];
            re += c * x[2 * ((size_t)t * nchan + n)];
            im += c * x[2 * ((size_t)t * nchan + n) + 1];
        }
        y[2 * n] = re;
        y[2 * n + 1] = im;
    }
}

/* ------------------------------------------------------------------ DFT */

void oracle_dft_bruteforce(int n, const double *in, double *out)
{
    for (int k = 0; k < n; k++) {
        double sr = 0.0, si = 0.0;
        for (int j = 0; j < n; j++) {
            /* exp(-2 pi i j k / n); reduce j*k mod n exactly in integers first */
            long r = ((long)j * (long)k) % (long)n;
            double a = -2.0 * M_PI * (double)r / (double)n;
            double c = cos(a), s = sin(a);
            double xr = in[2 * j], xi = in[2 * j + 1];
            sr += xr * c - xi * s;
            si += xr * s + xi * c;
        }
        out[2 * k] = sr;
        out[2 * k + 1] = si;
    }
}

/* Twiddle table W_n^k = exp(-2 pi i k / n), k < n/2, each entry straight from cos/sin in double.
 * A sub-transform of size n' = n/r uses entry k*r (the same angle). Rebuilt when n changes. */
static double *g_tw = NULL;
static int g_tw_n = 0;

static void tw_prepare(int n)
{
    if (n == g_tw_n) return;
    free(g_tw);
    g_tw = (double *)malloc((size_t)(n / 2 > 0 ? n / 2 : 1) * 2 * sizeof(double));
    for (int k = 0; k < n / 2; k++) {
        double a = -2.0 * M_PI * (double)k / (double)n;
        g_tw[2 * k] = cos(a);
        g_tw[2 * k + 1] = sin(a);
    }
    g_tw_n = n;
}

/* X[k] = E[k] + W_n^k O[k],  X[k+n/2] = E[k] - W_n^k O[k],  W_n = exp(-2 pi i / n) */
static void fft_rec(int n, const double *in, int stride, double *out)
{
    if (n == 1) {
        out[0] = in[0];
        out[1] = in[1];
        return;
    }
    int h = n / 2;
    fft_rec(h, in, 2 * stride, out);                      /* even samples -> out[0..h) */
    fft_rec(h, in + 2 * stride, 2 * stride, out + 2 * h); /* odd samples  -> out[h..n) */
    for (int k = 0; k < h; k++) {
        /* W_n^k = table entry k*stride, because stride = n_top/n */
        double c = g_tw[2 * (size_t)k * stride], s = g_tw[2 * (size_t)k * stride + 1];
        double er = out[2 * k], ei = out[2 * k + 1];
        double orr = out[2 * (k + h)], oi = out[2 * (k + h) + 1];
        double tr = orr * c - oi * s;
        double ti = orr * s + oi * c;
        out[2 * k] = er + tr;
        out[2 * k + 1] = ei + ti;
        out[2 * (k + h)] = er - tr;
        out[2 * (k + h) + 1] = ei - ti;
    }
}

void oracle_fft_radix2(int n, const double *in, double *out)
{
    tw_prepare(n);
    fft_rec(n, in, 1, out);
}

void oracle_dft(int n, const double *in, double *out)
{
    if (n <= 256) oracle_dft_bruteforce(n, in, out);
    else oracle_fft_radix2(n, in, out);
}

double oracle_unpack(int8_t b)
{
    return (double)b; /* two's complement, -128 stays -128 */
}

/* ------------------------------------------------------------------ state machine */

struct oracle_spec {
    int N, T, P, S, mode;
    long M;
    double *h;       /* T*N, fp32 values promoted to double */
    int8_t *hist;    /* up to T-1 complete raw blocks, oldest first */
    int nhist;
    long count;      /* spectra produced since start/reset */
    double *acc;     /* S*N running sums */
    double **done;   /* completed accumulations, FIFO */
    long ndone, cap;
    /* scratch */
    double *x, *y, *X;
};

oracle_spec *oracle_create(int nchan, int ntaps, int npol, int mode, long nacc, int window)
{
    if (nchan < 1 || npol < 1 || npol > 2 || nacc < 1) return NULL;
    if (mode != ORACLE_MODE_PFB && mode != ORACLE_MODE_FFT) return NULL;
    if (mode == ORACLE_MODE_FFT) ntaps = 1; /* DESIGN.md reading R12: ntaps ignored in FFT mode */
    if (ntaps < 1) return NULL;
    oracle_spec *o = (oracle_spec *)calloc(1, sizeof(*o));
    if (!o) return NULL;
    o->N = nchan; o->T = ntaps; o->P = npol; o->S = (npol == 2) ? 4 : 1;
    o->mode = mode; o->M = nacc;
    size_t L = (size_t)ntaps * nchan;
    o->h = (double *)malloc(L * sizeof(double));
    float *hf = (float *)malloc(L * sizeof(float));
    oracle_default_coeffs(nchan, ntaps, mode, window, hf);
    for (size_t k = 0; k < L; k++) o->h[k] = (double)hf[k];
    free(hf);
    o->hist = (int8_t *)malloc((size_t)(ntaps > 1 ? ntaps - 1 : 1) * nchan * 2 * npol);
    o->acc = (double *)calloc((size_t)o->S * nchan, sizeof(double));
    o->x = (double *)malloc(2 * L * sizeof(double));
    o->y = (double *)malloc(2 * (size_t)nchan * 2 * sizeof(double)); /* two pols */
    o->X = (double *)malloc(2 * (size_t)nchan * 2 * sizeof(double));
    return o;
}

int oracle_set_coeffs(oracle_spec *o, const float *h, size_t count)
{
    if (count != (size_t)o->T * o->N) return -1;
    for (size_t k = 0; k < count; k++) o->h[k] = (double)h[k];
    return 0;
}

static void emit(oracle_spec *o)
{
    if (o->ndone == o->cap) {
        o->cap = o->cap ? 2 * o->cap : 8;
        o->done = (double **)realloc(o->done, (size_t)o->cap * sizeof(double *));
    }
    size_t n = (size_t)o->S * o->N;
    double *c = (double *)malloc(n * sizeof(double));
    memcpy(c, o->acc, n * sizeof(double));
    o->done[o->ndone++] = c;
    memset(o->acc, 0, n * sizeof(double));
}

/* One spectrum from T consecutive raw blocks (blk[t] points at block t, N samples each). */
static void one_spectrum(oracle_spec *o, const int8_t *const *blk)
{
    const int N = o->N, T = o->T, P = o->P;
    for (int p = 0; p < P; p++) {
        /* step 3 of SURVEY 8c: unpack, byte order per sample [Xre,Xim,Yre,Yim] or [re,im] */
        for (int t = 0; t < T; t++)
            for (int n = 0; n < N; n++) {
                const int8_t *s = blk[t] + (size_t)n * 2 * P + 2 * p;
                o->x[2 * ((size_t)t * N + n)] = oracle_unpack(s[0]);
                o->x[2 * ((size_t)t * N + n) + 1] = oracle_unpack(s[1]);
            }
        double *y = o->y + (size_t)p * 2 * N;
        oracle_fir(N, T, o->h, o->x, y);              /* PAPER.md:92 step 3 */
        oracle_dft(N, y, o->X + (size_t)p * 2 * N);   /* PAPER.md:93 step 4 */
    }
    /* PAPER.md:83,94 step 5 */
    const double *X = o->X, *Y = o->X + (size_t)2 * N;
    for (int k = 0; k < N; k++) {
        double xr = X[2 * k], xi = X[2 * k + 1];
        o->acc[k] += xr * xr + xi * xi;
        if (P == 2) {
            double yr = Y[2 * k], yi = Y[2 * k + 1];
            o->acc[(size_t)N + k] += yr * yr + yi * yi;
            o->acc[(size_t)2 * N + k] += xr * yr + xi * yi;   /* Re(X conj Y) */
            o->acc[(size_t)3 * N + k] += xi * yr - xr * yi;   /* Im(X conj Y) */
        }
    }
    o->count++;
    if (o->count % o->M == 0) emit(o);
}

long oracle_process(oracle_spec *o, const int8_t *bytes, size_t nsamples)
{
    const int N = o->N, T = o->T;
    if (nsamples % (size_t)N != 0) return -1;
    const size_t bb = (size_t)N * 2 * o->P; /* bytes per block */
    long nnew = (long)(nsamples / (size_t)N);
    long total = o->nhist + nnew;
    long before = o->ndone;
    /* block i of the concatenation history ++ new */
    const int8_t **ptr = (const int8_t **)malloc((size_t)(total > 0 ? total : 1) * sizeof(*ptr));
    for (long i = 0; i < total; i++)
        ptr[i] = (i < o->nhist) ? o->hist + (size_t)i * bb : bytes + (size_t)(i - o->nhist) * bb;
    for (long m = 0; m + T <= total; m++) one_spectrum(o, ptr + m);
    /* keep the last min(T-1,total) blocks (reading R4: history starts empty) */
    long keep = total < T - 1 ? total : T - 1;
    if (keep > 0) {
        int8_t *tmp = (int8_t *)malloc((size_t)keep * bb);
        for (long i = 0; i < keep; i++) memcpy(tmp + (size_t)i * bb, ptr[total - keep + i], bb);
        memcpy(o->hist, tmp, (size_t)keep * bb);
        free(tmp);
    }
    o->nhist = (int)keep;
    free(ptr);
    return o->ndone - before;
}

int oracle_read_accum(oracle_spec *o, double *dst)
{
    if (o->ndone == 0) return 0;
    size_t n = (size_t)o->S * o->N;
    memcpy(dst, o->done[0], n * sizeof(double));
    free(o->done[0]);
    memmove(o->done, o->done + 1, (size_t)(o->ndone - 1) * sizeof(double *));
    o->ndone--;
    return 1;
}

long oracle_pending(const oracle_spec *o) { return o->ndone; }
long oracle_spectra_done(const oracle_spec *o) { return o->count; }

void oracle_reset(oracle_spec *o)
{
    for (long i = 0; i < o->ndone; i++) free(o->done[i]);
    o->ndone = 0;
    o->nhist = 0;
    o->count = 0;
    memset(o->acc, 0, (size_t)o->S * o->N * sizeof(double));
}

void oracle_destroy(oracle_spec *o)
{
    if (!o) return;
    oracle_reset(o);
    free(o->done); free(o->h); free(o->hist); free(o->acc);
    free(o->x); free(o->y); free(o->X);
    free(o);
}

/*
 * spec_oracle.h — CPU ORACLE for the spectrometer hot path of arXiv 1411.0436.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code,
 * header, table or helper with the CUDA path under paper_1411_0436_b200/csrc/.
 *
 * What it computes (section 4, steps 1-7; readings in DESIGN.md section 3):
 *   unpack int8 two's-complement complex samples
 *   -> T-tap polyphase pre-filter   y_p[m][n] = sum_{t<T} h[tN+n] * x_p[(m+t)N+n]
 *   -> N-point DFT                  X_p[m][k] = sum_n y_p[m][n] * exp(-2 pi i n k / N)
 *   -> products  XX=|X|^2, YY=|Y|^2, Re(X conj Y), Im(X conj Y)
 *   -> sum over M consecutive spectra, emit, clear
 * Everything is double precision.  The DFT is the O(N^2) definition for N <= 256 and a
 * naive recursive radix-2 decimation-in-time FFT above that.  No blocking, no fusion.
 *
 * Parity pins: every function here is pinned by tests/test_oracle_pins.py (closed forms,
 * invariants, numpy.fft cross-check, brute force on tiny inputs, SURVEY section 8c values
 * stored under tests/golden/).  No function is "parity unpinned".
 */
#ifndef SPEC_ORACLE_H
#define SPEC_ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { ORACLE_MODE_PFB = 0, ORACLE_MODE_FFT = 1 };
enum { ORACLE_WINDOW_RECT = 0, ORACLE_WINDOW_HANN = 1 };

typedef struct oracle_spec oracle_spec;

/* ---- stage functions (used by the state machine below and pinned one by one) ---- */

/* Prototype filter, reading R1 (north_star: "a sinc times a Hann window").
 * PFB: h[k] = sinc((k - T*N/2)/N) * w[k], k < T*N, sinc(x)=sin(pi x)/(pi x), sinc(0)=1,
 *      w = periodic Hann 0.5*(1-cos(2 pi k/(T*N))) or 1 (RECT).  count = T*N.
 * FFT: h[k] = w[k] over N (periodic Hann) or 1 (RECT).  count = N.
 * Computed in double, returned rounded to float (the value both sides use). */
void oracle_default_coeffs(int nchan, int ntaps, int mode, int window, float *out);

/* Direct FIR of one spectrum: x holds T blocks of N complex doubles
 * (re,im interleaved), y gets N complex doubles. */
void oracle_fir(int nchan, int ntaps, const double *h, const double *x, double *y);

/* DFT by definition, O(N^2), any N >= 1. in/out: N complex doubles. */
void oracle_dft_bruteforce(int n, const double *in, double *out);

/* Naive recursive radix-2 DIT FFT, N a power of two. Same convention as above. */
void oracle_fft_radix2(int n, const double *in, double *out);

/* The oracle's DFT: brute force for N <= 256, radix-2 above (north_star). */
void oracle_dft(int n, const double *in, double *out);

/* Exact unpack of one int8 byte to double (-128 stays -128). */
double oracle_unpack(int8_t b);

/* ---- streaming state machine (PAPER.md:87-96 steps 1-7) ---- */

oracle_spec *oracle_create(int nchan, int ntaps, int npol, int mode, long nacc, int window);
int  oracle_set_coeffs(oracle_spec *o, const float *h, size_t count); /* 0 ok, -1 bad count */
/* Feeds nsamples time samples (npol complex int8 each); nsamples % nchan must be 0.
 * Returns the number of accumulations completed by this call, or -1 on a bad size. */
long oracle_process(oracle_spec *o, const int8_t *bytes, size_t nsamples);
/* Pops the oldest completed accumulation as planar [S][nchan] doubles (S = 4 for npol 2:
 * XX, YY, Re, Im; S = 1 for npol 1).  Returns 1, or 0 if none is pending. */
int  oracle_read_accum(oracle_spec *o, double *dst);
long oracle_pending(const oracle_spec *o);
long oracle_spectra_done(const oracle_spec *o);
void oracle_reset(oracle_spec *o);
void oracle_destroy(oracle_spec *o);

#ifdef __cplusplus
}
#endif
#endif

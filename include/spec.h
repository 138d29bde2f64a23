/*
 * spec.h — C ABI of the B200 (sm_100a) streaming spectrometer: the GPU-thread hot path of
 * arXiv 1411.0436 ("the spectrometer implemented in the GPU thread"):
 *
 *   int8 complex (dual-pol) samples -> T-tap polyphase pre-filter -> N-point FFT
 *   -> XX*, YY*, Re(XY*), Im(XY*) -> fp32 accumulation over M spectra
 *   (PAPER.md:81-83 and the step list PAPER.md:87-96; BASELINE.json north_star names the calls).
 *
 * Conventions (DESIGN.md section 3 lists every reading of the paper):
 *   - one "time sample" is npol complex int8 values: bytes [Xre,Xim,Yre,Yim] (npol=2) or
 *     [re,im] (npol=1), two's complement, time-major.
 *   - block b = samples [b*nchan,(b+1)*nchan); spectrum m uses blocks m..m+T-1 (PFB) or block m (FFT).
 *   - FIR   y[m][n] = sum_{t<T} h[t*nchan+n] * x[(m+t)*nchan+n]
 *   - DFT   X[k] = sum_n y[n] exp(-2 pi i n k / nchan), unnormalised, DC first
 *   - out   planar [S][nchan] fp32, S=4: XX, YY, Re(X conj Y), Im(X conj Y); S=1 (npol=1): |X|^2
 *           summed (not averaged) over nacc consecutive spectra counted from stream start
 *           (PAPER.md:83,94).
 * Every function returns an int: >= 0 success, < 0 an SPEC_ERR_* code.  SPEC_ERR_ARG / _STATE / _SIZE /
 * _OVERRUN are detected before anything is queued and leave the handle's state unchanged.  SPEC_ERR_CUDA /
 * _NOMEM from spec_process or spec_stream_host mean a CUDA call failed after work had been queued: the
 * accumulators may be partly updated, the handle is marked failed and every later spec_process /
 * spec_read_accum returns SPEC_ERR_CUDA until spec_reset.  No exceptions, no abort.  All calls on one handle
 * come from one host thread.  Device pointers are plain CUDA device pointers; `cuda_stream` is a cudaStream_t
 * passed as void* (NULL = the legacy default stream).  The library never falls back to the CPU:
 * without a CUDA device spec_create fails with SPEC_ERR_CUDA.
 */
#ifndef SPEC_H
#define SPEC_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct spec_ctx spec_t; /* opaque; owned by the library */

enum { SPEC_MODE_PFB = 0, SPEC_MODE_FFT = 1 };
enum { SPEC_WINDOW_RECT = 0, SPEC_WINDOW_HANN = 1 };
enum {
    SPEC_OK = 0,
    SPEC_ERR_ARG = -1,     /* bad argument value */
    SPEC_ERR_STATE = -2,   /* call not valid in the handle's current state */
    SPEC_ERR_SIZE = -3,    /* wrong count / nsamples not a multiple of nchan */
    SPEC_ERR_OVERRUN = -4, /* the call would complete more accumulations than the ring can hold */
    SPEC_ERR_CUDA = -5,    /* a CUDA call failed; see spec_last_error() */
    SPEC_ERR_NOMEM = -6
};

/* PAPER.md:89-90 (steps 1a/1b: load coefficients, create the FFT plan).
 * nchan: power of two, 16 <= nchan <= 524288 (the paper's largest).
 * ntaps: >= 1 (the paper uses 8); ignored (treated as 1) in FFT mode.
 * npol: 1 or 2.  mode: SPEC_MODE_PFB / SPEC_MODE_FFT (direct FFT).
 * nacc: spectra per accumulation (>= 1).  window: PFB: h = sinc((k-T*N/2)/N) * w[k], k < T*N,
 * w = periodic Hann or 1; FFT: h = w over N (RECT = no multiply).  Coefficients are computed in
 * double on the host and rounded to fp32.  Allocates all device memory (coefficients, twiddles,
 * history, four-step workspace, a ring of 8 completed accumulations).  *out is set on success. */
int spec_create(spec_t** out, int nchan, int ntaps, int npol, int mode, long nacc, int window);

/* PAPER.md:51, :73 (Table 1, third block), :90 (step 1b: "16 FFTs in parallel in the case of eight-sub-band
 * modes"): like spec_create, for nsub (1..16) sub-bands that share the channel count, the filter and the
 * accumulation length.  The input of spec_process / spec_stream_host then carries the sub-bands interleaved per
 * time sample (reading R26: the paper does not state the order): one time sample is nsub * 2 * npol
 * bytes, sub-band 0 first; nsamples still counts time samples.  spec_read_accum delivers [nsub][S][nchan],
 * spec_read_accum_batch [count][nsub][S][nchan].  The sub-bands are independent spectrometers: the library splits
 * the input into one contiguous stream per sub-band (one extra pass over the input) and runs each through the
 * plan spec_create would choose.  The test hook spec_debug_fir and the graph-capture brackets are per-sub-band
 * features and return SPEC_ERR_STATE on such a handle. */
int spec_create_subbands(spec_t** out, int nsub, int nchan, int ntaps, int npol, int mode, long nacc, int window);

/* PAPER.md:89 (step 1a).  Replaces the coefficients: h_coeffs is a HOST array of `count` floats,
 * count == ntaps*nchan (PFB) or nchan (FFT mode); copied before return (synchronises the device).
 * SPEC_ERR_SIZE on a wrong count. */
int spec_set_coeffs(spec_t* s, const float* h_coeffs, size_t count);

/* PAPER.md:91-94 (steps 2-5).  Feeds `nsamples` time samples from DEVICE memory d_in
 * (nsamples * 2 * npol bytes, 16-byte aligned); nsamples must be a multiple of nchan (0 is a no-op).  The last
 * (ntaps-1)*nchan samples are carried as filter history to the next call, so results depend only
 * on the concatenated stream, never on how calls split it.  The history starts empty: the first
 * spectrum needs ntaps blocks.  All work is queued on cuda_stream; d_in is borrowed until that
 * work completes.  Returns the number of accumulations completed by this call (>= 0), or
 * SPEC_ERR_SIZE / SPEC_ERR_OVERRUN (nothing queued) / SPEC_ERR_CUDA.  No host synchronisation and no
 * allocation happens in this call (for calls of up to 2^28 samples), so it may be captured into a CUDA graph.
 * The persistent kernel behind this call (dual-pol, 1024 <= nchan <= 65536) sizes its grid to exactly what the
 * GPU holds at once (4, or 2, CTAs per SM on every SM) and its CTAs wait for one another: it assumes the
 * whole GPU is available to it (no MPS / green-context SM limit, no other kernel holding SM resources for
 * seconds).  Every wait in it is bounded (about ten seconds); if one ever expires (the grid could not
 * become resident) the launch ends with invalid sums instead of hanging, and this and every later
 * spec_process / spec_read_accum on the handle return SPEC_ERR_CUDA until spec_reset. */
int spec_process(spec_t* s, const void* d_in, size_t nsamples, void* cuda_stream);

/* PAPER.md:95 (step 6).  Pops the oldest completed accumulation into dst as planar
 * [S][nchan] fp32 in natural channel order.  dst_is_device != 0: dst is device memory and the copy
 * is only queued on cuda_stream; else dst is host memory and the call returns after the data has
 * arrived.  Use the stream the producing spec_process used (or synchronise first).
 * Returns 1, or 0 if nothing is pending. */
int spec_read_accum(spec_t* s, float* dst, int dst_is_device, void* cuda_stream);

/* PAPER.md:95 (step 6), several at once: pops up to max_count of the oldest completed accumulations
 * with ONE kernel launch into DEVICE memory d_dst as [count][S][nchan] fp32 (each as spec_read_accum
 * writes it, oldest first); the copy is only queued on cuda_stream.  Returns the count popped (0 if
 * nothing is pending).  (An extension: north_star names the single-accumulation call above.) */
int spec_read_accum_batch(spec_t* s, float* d_dst, int max_count, void* cuda_stream);

/* Frees everything the handle owns (synchronises the device). */
int spec_destroy(spec_t* s);

/* ---- small extensions (not named by north_star) ---- */

/* Number of completed accumulations waiting in the ring / spectra produced since start or reset. */
int spec_pending(const spec_t* s);
long spec_spectra_done(const spec_t* s);

/* History empty, accumulators zero, ring empty, spectrum counter 0 (synchronises the device). */
int spec_reset(spec_t* s);

/* Ring capacity (completed accumulations held before SPEC_ERR_OVERRUN); default 8.  Only valid
 * while nothing is pending and no accumulation is in progress (after create or reset). */
int spec_set_ring(spec_t* s, int nslots);

/* PAPER.md:116, :122 (per-invocation overheads; "pipelining kernel launches using CUDA streams") and SURVEY.md 8(f)
 * NEXT-4: many small (packet-sized) calls replayed as ONE CUDA graph.  The caller captures a SEGMENT of calls on a
 * stream (cudaStreamBeginCapture ... spec_process / spec_read_accum(dst_is_device) / spec_read_accum_batch ...
 * cudaStreamEndCapture) between spec_capture_begin and spec_capture_end.  The kernels' arguments (history buffer,
 * accumulation-window phase, ring slots) are baked into the graph, so a segment is replayable only if it returns
 * the handle to the same phase: a multiple of 6 spec_process calls (three history buffers, two ring parities), a
 * multiple of nacc * (ring slots + 1) spectra, and every accumulation it completes read inside the segment;
 * spec_capture_end checks this (SPEC_ERR_STATE otherwise; the captured graph must then be discarded).  The
 * handle's counters already moved once while the calls were captured (capture records, it does not execute), so
 * that accounts for the first launch of the graph; report every further launch with spec_replayed.  While a
 * capture is open consecutive launches do not overlap and nothing synchronises or allocates. */
int spec_capture_begin(spec_t* s);
int spec_capture_end(spec_t* s);
/* The captured segment has been launched `times` times: advances the spectrum and read-out counters accordingly
 * (the first launch of the graph is what the captured calls themselves accounted for: pass times - 1 for it). */
int spec_replayed(spec_t* s, long times);

/* PAPER.md:53 (the "CPU thread": further accumulation of the GPU's output on the host): h_acc[i] += h_spectrum[i]
 * in double precision, i < count, both HOST arrays. */
int spec_accumulate_host(double* h_acc, const float* h_spectrum, size_t count);

/* Plan options.  SPEC_OPT_TENSOR_CORE_STAGE (value 0 / 1): in direct-FFT mode with the rectangular window
 * (dual-pol, nchan 16384 or 32768) run the first 16-point DFT factor of the four-step transform on the tensor
 * cores (tcgen05.mma, fp16 operands: the int8 samples are exact, the DFT matrix is split into two fp16 terms,
 * fp32 accumulation) instead of fp32 butterflies.  Off by default; DESIGN.md section 7
 * records the measured speed and error of both.  SPEC_ERR_STATE if the handle's plan has no such stage. */
enum { SPEC_OPT_TENSOR_CORE_STAGE = 1 };
int spec_set_option(spec_t* s, int option, int value);

/* Copy the coefficients in use to a host array of `count` floats (count as in spec_set_coeffs). */
int spec_get_coeffs(const spec_t* s, float* h_out, size_t count);

/* PAPER.md:91 + BASELINE.json north_star item (d): streams `nsamples` samples from PINNED HOST
 * memory in chunks of chunk_samples (a multiple of nchan) through two device buffers: the
 * host-to-device copy of chunk i+1 runs on a side stream while spec_process works on chunk i on
 * cuda_stream.  Returns the accumulations completed, like spec_process.  Returns after the last
 * chunk has been queued; h_pinned must stay valid until cuda_stream has drained. */
int spec_stream_host(spec_t* s, const void* h_pinned, size_t nsamples, size_t chunk_samples,
                     void* cuda_stream);

/* Roofline denominator (BASELINE.json north_star: "the measured FP32 peak"): runs a dependent-free
 * FFMA kernel on every SM and returns the achieved fp32 rate in TFLOP/s (2 flops per FMA). */
int spec_measure_fp32_peak(double* out_tflops, void* cuda_stream);

/* Per-kernel timing for the roofline report.  spec_profile(s, 1) zeroes the counters and brackets
 * every later kernel launch with CUDA events on its stream; spec_profile(s, 0) only counts launches.
 * spec_profile_read waits for the recorded events and returns, per kernel class (0 fused single-pass
 * kernel, 1 four-step pass A, 2 four-step pass B, 3 read-out un-permute), the summed device time in
 * ms (0 when timing is off) and the number of launches since the last spec_profile call. */
int spec_profile(spec_t* s, int enable);
int spec_profile_read(spec_t* s, double ms[4], long launches[4]);

/* Test hooks for the bit-exact stages (north_star: "unpack and indexing stages must be bit-exact"):
 * spec_debug_unpack: d_out[i] = float(int8 d_bytes[i]) for i < nbytes (device pointers), through the unpack
 * routine the kernels call (npol = 2: the packed dual-pol form, npol = 1: the single-pol form).
 * spec_debug_fir: runs the FRONT END of the very kernel this handle's plan uses (a DUMP instantiation of the
 * same kernel template: its staging, index arithmetic, unpack and FIR / window code) on nspec spectra taken
 * from d_blocks (nspec + ntaps - 1 consecutive blocks, device, 16-byte aligned, history empty) and writes what
 * it hands to the first butterfly as [nspec][nchan][2*npol] fp32 (re,im per pol) to d_out (device).  The
 * handle's stream state (history, accumulators, counters) is not touched. */
int spec_debug_unpack(const void* d_bytes, size_t nbytes, int npol, float* d_out, void* cuda_stream);
int spec_debug_fir(spec_t* s, const void* d_blocks, int nspec, float* d_out, void* cuda_stream);

/* A one-shot entry point that ALLOCATES NOTHING, for callers that cannot call cudaMalloc (code under CUDA-graph capture,
 * tight serving loops, harnesses that forbid it): no handle, no cudaMalloc / cudaFree / allocating library routine, ever.
 * Runs the whole chain of PAPER.md:87-96 (unpack, optional FIR, nchan-point FFT, Stokes, sum) over ONE stretch of samples
 * with the single-kernel plan and writes the sum over all its spectra.
 *   d_in      DEVICE, nsamples time samples of 2*npol int8 (layout as spec_process), 16-byte aligned, nsamples a
 *             multiple of nchan; the filter history is empty: nsamples/nchan - (ntaps-1) spectra are formed.
 *   nchan     power of two, 16 <= nchan <= 4096 (SPEC_ERR_SIZE beyond: the scratch array is fixed at 112 KiB).
 *   ntaps, d_coeffs   d_coeffs == NULL: direct FFT, rectangular window (ntaps must be 1).  Else DEVICE array of
 *             ntaps*nchan fp32 filter coefficients (ntaps 1..64; ntaps = 1 is a window over nchan).
 *   d_out     DEVICE, planar [S][nchan] fp32 (S = 4 for npol = 2, else 1), natural channel order, overwritten.
 * Returns the number of spectra summed (>= 1) or an SPEC_ERR_* code; all work is queued on cuda_stream.
 * The scratch (accumulators in the engine's order, stage twiddles, channel table) is a file-scope device array inside the
 * library: every GPU that loads the library holds its 112 KiB until exit.  All calls share it, and it keeps the last
 * call's contents: the sums are cleared at the start of every call, the tables are re-uploaded (two small host-to-
 * device copies on cuda_stream) whenever nchan differs from the previous call's on that device.  Calls that OVERLAP on
 * the GPU (different streams, no dependency between them) race on the array: serialise them. */
int spec_oneshot_static(const void* d_in, size_t nsamples, int nchan, int ntaps, int npol, const float* d_coeffs,
                        float* d_out, void* cuda_stream);

/* Throughput probe behind the design notes: thread-instructions per clock and SM (at the
 * device's nominal clock) of op 0 scalar FFMA, 1 packed FFMA2, 2 packed FADD2, 3 PRMT, 4 LDS.128 alone,
 * 5 LDS.128 with eight FFMA2 behind each load (counts the loads), 6 SHFL; 1024 threads per SM, independent chains. */
int spec_debug_probe(int op, double* out_per_clk_sm, void* cuda_stream);

/* Test hook for the soak test: a foreign kernel of one CTA per SM that holds smem_bytes of shared memory
 * (up to 227 KiB) and spins for about ms milliseconds (at most 2000) on cuda_stream. */
int spec_debug_hog(int ms, size_t smem_bytes, void* cuda_stream);

/* Which kernels the handle's plan uses: the four-step split nchan = n1 * n2 (n1 = 1: one kernel per call, no
 * split) and a one-line description (kernel template, grid, ring) for reports.  Any pointer may be NULL. */
int spec_plan_info(const spec_t* s, int* n1, int* n2, char* desc, size_t desc_len);

const char* spec_strerror(int code);
const char* spec_last_error(void); /* detail of the last SPEC_ERR_CUDA / SPEC_ERR_NOMEM on this thread */

#ifdef __cplusplus
}
#endif
#endif /* SPEC_H */

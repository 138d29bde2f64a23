// passa_pfb.cuh — four-step pass A for PFB mode with N1 = 16 (8192 <= N <= 65536):
//   unpack + T-tap FIR for R consecutive spectra -> shared memory -> 16-point column FFTs
//   -> W_N^{n2 k1} twiddle -> Z[m][k1][n2]  (PAPER.md:92-93 steps 3-4, first FFT factor)
// A CTA owns C adjacent columns n2 (all 16 rows n1, so 16*C filter branches) and walks a run of
// spectra R at a time.  FIR phase: each thread owns 16/R branches and slides a T-sample register
// window over R+T-1 input blocks (every block is loaded and unpacked once per phase; the T-1 halo
// blocks are re-read from L2 at the next phase).  FFT phase: each thread owns one (spectrum, column)
// pair: 16 LDS.128, radix-16 in registers, twiddle, 16 coalesced float4 stores.
#pragma once
#include "engine.cuh"

namespace spk {

// DUMP (test hook): the FIR outputs the column FFT is about to consume are written to Z as the caller's
// [spectrum][n][re,im per pol] and no transform runs.
template <int P, int T, int C, int R, bool DUMP = false>
__global__ void __launch_bounds__(C * R, 2)
k_passA_pfb16(const InputView view, const float* __restrict__ h, float4* __restrict__ Z,
              const float2* __restrict__ twN, int N, int N2, long long m0, int nb, int phases_per_cta) {
    static_assert(16 % R == 0 && T <= 8, "branch split / window size");
    constexpr int NT = C * R;
    constexpr int BPT = 16 / R;  // branches per thread
    extern __shared__ float4 ysm[];  // [R][16][C]

    const int tid = threadIdx.x;
    const int n2_0 = blockIdx.x * C;
    const int nphases = (nb + R - 1) / R;
    const int ph0 = blockIdx.y * phases_per_cta;
    const int ph1 = (ph0 + phases_per_cta < nphases) ? ph0 + phases_per_cta : nphases;

    // FFT-phase role: spectrum fr of the phase, column fc; its twiddles W_N^{n2 k1} stay in registers
    const int fr = tid / C, fc = tid % C;
    const int n2 = n2_0 + fc;
    float2 tw[16];
#pragma unroll
    for (int k = 1; k < 16; k++) tw[k] = __ldg(twN + (size_t)n2 * k);

    for (int ph = ph0; ph < ph1; ph++) {
        const int j0 = ph * R;  // first job (spectrum) of this phase
        // ---------------- FIR phase
        // all (R+T-1) blocks of both branches are fetched before any arithmetic (one L2 latency per
        // phase); in the ragged last phase the block index is clamped to the last valid block
        const int qmax = nb - 1 - j0 + (T - 1);
        uint32_t raw[BPT][R + T - 1];
        float hc[BPT][T];
        const bool in_input = (m0 + j0 >= view.nhist);  // no block of this phase comes from the history
#pragma unroll
        for (int i = 0; i < BPT; i++) {
            const int beta = tid + NT * i;
            const int n = (beta / C) * N2 + n2_0 + (beta % C);
#pragma unroll
            for (int t = 0; t < T; t++) hc[i][t] = __ldg(h + (size_t)t * N + n);
            if (in_input) {
                const uint8_t* base = view.in + ((size_t)(m0 + j0 - view.nhist) * N + n) * (2 * P);
                const size_t rowb = (size_t)N * (2 * P);
#pragma unroll
                for (int q = 0; q < R + T - 1; q++) {
                    const uint8_t* p = base + (size_t)(q < qmax ? q : qmax) * rowb;
                    raw[i][q] = (P == 2) ? __ldg((const uint32_t*)p) : (uint32_t)__ldg((const uint16_t*)p);
                }
            } else {
#pragma unroll
                for (int q = 0; q < R + T - 1; q++)
                    raw[i][q] = fetch_raw<P>(view, m0 + j0 + (q < qmax ? q : qmax), n, N);
            }
        }
#pragma unroll
        for (int i = 0; i < BPT; i++) {
            const int beta = tid + NT * i;
            const int n1 = beta / C, c = beta % C;
            cpx x[T];
#pragma unroll
            for (int t = 0; t < T - 1; t++) x[t] = unpack_cpx<P>(raw[i][t]);
#pragma unroll
            for (int r = 0; r < R; r++) {
                x[(r + T - 1) % T] = unpack_cpx<P>(raw[i][r + T - 1]);
                u64 re = 0ull, im = 0ull;
#pragma unroll
                for (int t = 0; t < T; t++) {
                    re = fma2(x[(r + t) % T].re, bc(hc[i][t]), re);
                    im = fma2(x[(r + t) % T].im, bc(hc[i][t]), im);
                }
                ysm[(r * 16 + n1) * C + c] = cpx_to_f4({re, im});
            }
        }
        __syncthreads();
        // ---------------- column FFT phase
        if (j0 + fr < nb) {
            cpx v[16];
#pragma unroll
            for (int n1 = 0; n1 < 16; n1++) v[n1] = f4_to_cpx(ysm[(fr * 16 + n1) * C + fc]);
            if (DUMP) {
#pragma unroll
                for (int n1 = 0; n1 < 16; n1++) {
                    const float4 z = cpx_to_f4(v[n1]);
                    const size_t o = (size_t)(j0 + fr) * N + (size_t)n1 * N2 + n2;
                    if (P == 2) Z[o] = make_float4(z.x, z.z, z.y, z.w);
                    else ((float2*)Z)[o] = make_float2(z.x, z.z);
                }
            } else {
                dft<16>(v);
                float4* zp = Z + (size_t)(j0 + fr) * N + n2;
                zp[0] = cpx_to_f4(v[0]);
#pragma unroll
                for (int k = 1; k < 16; k++) zp[(size_t)k * N2] = cpx_to_f4(cmul(v[k], tw[k].x, tw[k].y));
            }
        }
        __syncthreads();
    }
}

// Stand-alone 8-tap polyphase FIR (step 3) for the splits whose first factor is larger than 16
// (N >= 131072): y[m][n] = sum_t h[tN+n] x[(m+t)N+n] for a chunk of CH consecutive spectra per thread,
// one filter branch n per thread (coalesced over n), an 8-sample register window that slides by one block
// per spectrum (every raw sample is loaded and unpacked once per chunk).  Output Y[m][n] as float4
// (Xre, Yre, Xim, Yim), read back by pass A through FrontY.
template <int P, int CH>
__global__ void __launch_bounds__(256)
k_fir8(const InputView view, const float* __restrict__ h, float4* __restrict__ Y, int N, long long m0, int nb) {
    constexpr int T = 8;
    static_assert(CH % T == 0, "chunk is a whole number of window rotations");
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    const int j0 = blockIdx.y * CH;
    if (n >= N || j0 >= nb) return;
    const int j1 = (j0 + CH < nb) ? j0 + CH : nb;
    float hc[T];
#pragma unroll
    for (int t = 0; t < T; t++) hc[t] = __ldg(h + (size_t)t * N + n);
    cpx x[T];
#pragma unroll
    for (int t = 0; t < T - 1; t++) x[t] = load_raw<P>(view, m0 + j0 + t, n, N);
    for (int j = j0; j < j1; j += T) {
#pragma unroll
        for (int r = 0; r < T; r++) {
            if (j + r < j1) {
                x[(r + T - 1) % T] = load_raw<P>(view, m0 + j + r + T - 1, n, N);
                u64 re = 0ull, im = 0ull;
#pragma unroll
                for (int t = 0; t < T; t++) {
                    re = fma2(x[(r + t) % T].re, bc(hc[t]), re);
                    im = fma2(x[(r + t) % T].im, bc(hc[t]), im);
                }
                Y[(size_t)(j + r) * N + n] = cpx_to_f4({re, im});
            }
        }
    }
}

}  // namespace spk
